// Immersed-boundary kernels: rigid-rotation kinematics (a1, a2), bins + active-cell mask (a3),
// interpolation (a5), direct-forcing correction (a6), spreading (a7).  Section 3 of the paper
// with the readings R6-R14 of DESIGN.md.
//
// Marker position is kept as (integer cell, fractional offset in [0,1)) per axis, so the delta
// kernel arguments never lose bits to the magnitude of the coordinate.
#pragma once
#include "lbm_kernels.cuh"

namespace lbmk {

// per-body constants (host-filled, fp64) and per-step rotation tables (device-filled)
struct BodyDef {
    double omega, ax, ay, az;      // unit axis
    int ci[3];                     // centre = ci + cf, cf in [0,1)
    float cf[3];
};
struct BodyStep {
    float R[9];    // R(omega (n+1))
    float dR[9];   // R(omega (n+1)) - R(omega n), formed in fp64 (R12)
};

struct MarkerIn {                  // original (caller) order
    const float4 *qs;              // (rest position relative to the body centre p_k - c (fp64 -> fp32), area s(k))
    const float4 *vb;              // (extra velocity vel_k (R14), body id as int bits)
    const int *body;               // body id once more, for the kernels that read in caller order
    int n;                         // two 16-byte records per marker: the gather by the sort permutation touches
};                                 // two sectors per marker instead of eight

// a1: Rodrigues rotation tables of every body for step n -> n+1, in fp64 (R12, R13).
// Also re-arms the per-step device counters of the marker set being prepared.  step_offset = 1
// when the tables of the NEXT step are prepared while the current one is still running.
__global__ void k_kinematics(const BodyDef *__restrict__ defs, BodyStep *__restrict__ out, int nbodies,
                             const long long *__restrict__ step_ctr, int step_offset, int *__restrict__ counters,
                             int n_counters)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n_counters) counters[b] = 0;
    if (b >= nbodies) return;
    const BodyDef d = defs[b];
    const double n = (double)(*step_ctr + step_offset);
    double R1[9], R0[9];
    for (int which = 0; which < 2; ++which) {
        const double th = d.omega * (n + (which == 0 ? 1.0 : 0.0));
        double s, c;
        sincos(th, &s, &c);
        const double v = 1.0 - c;
        double *R = which == 0 ? R1 : R0;
        R[0] = c + d.ax * d.ax * v;        R[1] = d.ax * d.ay * v - d.az * s; R[2] = d.ax * d.az * v + d.ay * s;
        R[3] = d.ay * d.ax * v + d.az * s; R[4] = c + d.ay * d.ay * v;        R[5] = d.ay * d.az * v - d.ax * s;
        R[6] = d.az * d.ax * v - d.ay * s; R[7] = d.az * d.ay * v + d.ax * s; R[8] = c + d.az * d.az * v;
    }
    BodyStep o;
    for (int j = 0; j < 9; ++j) { o.R[j] = (float)R1[j]; o.dR[j] = (float)(R1[j] - R0[j]); }
    out[b] = o;
}

// Peskin 4-point kernel (R6): the four distances 1+f, f, 1-f, 2-f of a point at c + f to the
// cells c-1 .. c+2 share one square root, because 1 + 4r - 4r^2 at r = f or 1-f and -7 + 12r - 4r^2
// at r = 1+f or 2-f all equal 1 + 4f(1 - f).
__device__ __forceinline__ float peskin_root(float f) { return sqrtf(fmaf(4.0f * f, 1.0f - f, 1.0f)); }

struct Placed {
    int cx, cy, cz;      // owning cell = floor(position), wrapped on periodic axes
    float fx, fy, fz;    // position - cell, in [0,1)
    bool bad;            // stencil would cross a wall face (R17); cell clamped
};

__device__ __forceinline__ void place_axis(float d, int ci, int n, int wall, int &c, float &f, bool &bad)
{
    const float fl = floorf(d);
    f = d - fl;
    c = ci + (int)fl;
    if (f >= 1.0f) { f = 0.0f; c += 1; }       // d = -tiny rounds d - floor(d) up to 1
    if (wall) {
        if (c < 1 || c > n - 3) { bad = true; c = min(max(c, 1), n - 3); }
    } else {
        c %= n;
        if (c < 0) c += n;
    }
}

// a2: x_k = c + R (p_k - c) as (cell, fraction).  Used by BOTH the key kernel and the gather kernel
// so the two always agree on the owning cell.
__device__ __forceinline__ Placed place_marker(const BodyDef &d, const BodyStep &t, float qx, float qy, float qz,
                                               const Geom &g)
{
    Placed p;
    p.bad = false;
    const float dx = fmaf(t.R[0], qx, fmaf(t.R[1], qy, fmaf(t.R[2], qz, d.cf[0])));
    const float dy = fmaf(t.R[3], qx, fmaf(t.R[4], qy, fmaf(t.R[5], qz, d.cf[1])));
    const float dz = fmaf(t.R[6], qx, fmaf(t.R[7], qy, fmaf(t.R[8], qz, d.cf[2])));
    place_axis(dx, d.ci[0], g.nx, g.wallx, p.cx, p.fx, p.bad);
    place_axis(dy, d.ci[1], g.ny, g.wally, p.cy, p.fy, p.bad);
    place_axis(dz, d.ci[2], g.nz, g.wallz, p.cz, p.fz, p.bad);
    return p;
}

// a2: cell key of every marker (original order): key = (cz ny + cy) nx + cx  (O3).
__global__ void __launch_bounds__(256)
k_marker_keys(MarkerIn m, const BodyDef *__restrict__ defs, const BodyStep *__restrict__ tabs, Geom g,
              unsigned *__restrict__ keys, int *__restrict__ status, long long *__restrict__ advance_ctr)
{
    // advance_ctr != NULL: this launch follows the only k_kinematics of its step graph in the same chain, so the
    // device-side time-step counter (read by k_kinematics alone) can advance here instead of in a kernel of its own
    if (advance_ctr && blockIdx.x == 0 && threadIdx.x == 0) *advance_ctr += 1;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m.n) return;
    const int b = m.body[k];
    const float4 q = __ldg(m.qs + k);
    const Placed p = place_marker(defs[b], tabs[b], q.x, q.y, q.z, g);
    if (p.bad) *status = 1;
    keys[k] = (unsigned)((p.cz * g.ny + p.cy) * g.nx + p.cx);
}

// Peskin 4-point weights of the cells c-1, c, c+1, c+2 for a point at c + f, 0 <= f < 1 (R6).
// The four distances 1+f, f, 1-f, 2-f share one square root: 1 + 4r - 4r^2 at r = f or 1-f and
// -7 + 12r - 4r^2 at r = 1+f or 2-f all equal 1 + 4f - 4f^2.
__device__ __forceinline__ void peskin4(float f, float (&w)[4])
{
    const float q = peskin_root(f);
    const float a = 3.0f - 2.0f * f, b = 1.0f + 2.0f * f;
    w[0] = 0.125f * (a - q);
    w[1] = 0.125f * (a + q);
    w[2] = 0.125f * (b + q);
    w[3] = 0.125f * (b - q);
}

// per-marker state in SORTED order
struct MarkerSorted {
    float4 *fs;     // (fx, fy, fz, s)
    float4 *wx;     // the four x weights w(x_k - X), X = cx-1 .. cx+2       (unfused comparison path only, else NULL)
    float *wyz;     // [16] per marker: w_y(jy) w_z(jz) at index jy*4+jz     (unfused comparison path only, else NULL)
                    // sg.w and du.w carry the marker's cell x index (int bits) for the chunk sweep
    float4 *uk;     // prescribed velocity u_k, w unused
    float4 *sg;     // s * g^m(k)   (what the U update spreads, P:98 + R8)   (comparison paths only, else NULL)
    float4 *du;     // Delta u(k)
};

// a2 (second half): gather into sorted order; u_k = dR (p_k - c) + vel_k (chord velocity, R12).
__global__ void __launch_bounds__(256)
k_marker_gather(MarkerIn m, const BodyDef *__restrict__ defs, const BodyStep *__restrict__ tabs, Geom g,
                const int *__restrict__ perm, MarkerSorted out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m.n) return;
    const int k = perm[i];
    const float4 q = __ldg(m.qs + k), v = __ldg(m.vb + k);
    const int b = __float_as_int(v.w);
    const BodyStep t = tabs[b];
    const float qx = q.x, qy = q.y, qz = q.z;
    const Placed p = place_marker(defs[b], t, qx, qy, qz, g);
    out.fs[i] = make_float4(p.fx, p.fy, p.fz, q.w);

    const float ux = fmaf(t.dR[0], qx, fmaf(t.dR[1], qy, fmaf(t.dR[2], qz, v.x)));
    const float uy = fmaf(t.dR[3], qx, fmaf(t.dR[4], qy, fmaf(t.dR[5], qz, v.y)));
    const float uz = fmaf(t.dR[6], qx, fmaf(t.dR[7], qy, fmaf(t.dR[8], qz, v.z)));
    out.uk[i] = make_float4(ux, uy, uz, 0.f);
    out.du[i] = make_float4(0.f, 0.f, 0.f, __int_as_float(p.cx));
    if (!out.sg) return;                             // the fused tile pass (mdf_kernels.cuh) needs no tables
    out.sg[i] = make_float4(0.f, 0.f, 0.f, __int_as_float(p.cx));
    if (!out.wx) return;
    // per-step weight tables of the round-1 chunk sweep (the position does not change during the MDF loop)
    float wx[4], wy[4], wz[4];
    peskin4(p.fx, wx);
    peskin4(p.fy, wy);
    peskin4(p.fz, wz);
    out.wx[i] = make_float4(wx[0], wx[1], wx[2], wx[3]);
    float4 *w16 = reinterpret_cast<float4 *>(out.wyz + (size_t)i * 16);
#pragma unroll
    for (int jy = 0; jy < 4; ++jy) w16[jy] = make_float4(wy[jy] * wz[0], wy[jy] * wz[1], wy[jy] * wz[2], wy[jy] * wz[3]);
}

__device__ __forceinline__ void key_to_cell(unsigned key, const Geom &g, int &cx, int &cy, int &cz)
{
    const int row = (int)(key / (unsigned)g.nx);
    cx = (int)key - row * g.nx;
    cz = row / g.ny;
    cy = row - cz * g.ny;
}

__device__ __forceinline__ int wrap(int i, int n)
{
    return i < 0 ? i + n : (i >= n ? i - n : i);
}

// a3: bins and active cells.  The first marker of every occupied cell ("bin head") records its
// sorted index in the dense cell -> first-marker map and marks the 4x4x4 cells of its stencil in
// the active-cell bitmask (one bit per cell, 32 consecutive x per word).
__global__ void __launch_bounds__(256)
k_bins(const unsigned *__restrict__ skey, int n, Geom g, int *__restrict__ bin_first, unsigned *__restrict__ amask)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool head = false;
    int cx = 0, cy = 0, cz = 0;
    if (i < n) {
        const unsigned key = skey[i];
        head = (i == 0) || (skey[i - 1] != key);
        if (head) {
            bin_first[key] = i;
            key_to_cell(key, g, cx, cy, cz);
        }
    }
    // the four x cells cx-1..cx+2 fall into at most two words, or three when they wrap on a lattice whose last word
    // holds one or two cells (nx % 32 = 1, 2: e.g. nx = 65, cells 63 | 64 | 0, 1)
#pragma unroll 1
    for (int r = 0; r < 16; ++r) {
        const int y = wrap(cy - 1 + (r & 3), g.ny);
        const int z = wrap(cz - 1 + (r >> 2), g.nz);
        const int rowbase = (z * g.ny + y) * g.nxw;
        int w0 = -1, w1 = -1, w2 = -1;
        unsigned b0 = 0, b1 = 0, b2 = 0;
        if (head) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int x = wrap(cx - 1 + j, g.nx);
                const int w = rowbase + (x >> 5);
                const unsigned bit = 1u << (x & 31);
                if (w0 < 0 || w == w0) { w0 = w; b0 |= bit; }
                else if (w1 < 0 || w == w1) { w1 = w; b1 |= bit; }
                else { w2 = w; b2 |= bit; }
            }
        }
        if (w0 >= 0) atomicOr(amask + w0, b0);
        if (w1 >= 0) atomicOr(amask + w1, b1);
        if (w2 >= 0) atomicOr(amask + w2, b2);
    }
}

// Undo what the previous preparation of this marker set left in the dense maps (bitmask words, chunk
// registrations, cell -> first-marker entries), so none of them needs a full memset per step.
__global__ void __launch_bounds__(256)
k_clear_prev(const unsigned *__restrict__ skey_prev, const int *__restrict__ n_prev, int *__restrict__ bin_first,
             unsigned *__restrict__ amask, const int *__restrict__ words, const int *__restrict__ n_words,
             int *__restrict__ chunk_of, const int *__restrict__ chunk_slot, const int *__restrict__ n_chunks, int cap,
             unsigned *__restrict__ tile_mask, const int *__restrict__ tile_slot, const int *__restrict__ n_tiles,
             int tile_cap, const int *__restrict__ ovf_slot, const int *__restrict__ n_ovf, int ovf_cap, int n_tile_slots)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const int np = *n_prev, nw = *n_words, nc = min(*n_chunks, cap);
    if (bin_first) for (int i = tid; i < np; i += stride) bin_first[skey_prev[i]] = -1;
    for (int i = tid; i < nw; i += stride) amask[words[i]] = 0u;
    for (int c = tid; c < nc; c += stride) chunk_of[chunk_slot[c]] = -1;
    const int nt = min(*n_tiles, tile_cap);
    for (int c = tid; c < nt; c += stride) tile_mask[tile_slot[c]] = 0u;
    // tile slots that were registered without a footprint (tile table overflow) are listed apart; when even that
    // list overflowed, every slot is cleared
    const int no = *n_ovf;
    if (no <= ovf_cap) { for (int c = tid; c < no; c += stride) tile_mask[ovf_slot[c]] = 0u; }
    else { for (int c = tid; c < n_tile_slots; c += stride) tile_mask[c] = 0u; }
}

// device scalars: mode bit 0: step_ctr = step; bit 1: n_prev = n_prev_val; bit 2: step_ctr += 1
__global__ void k_set_scalars(long long *step_ctr, long long step, int *n_prev, int n_prev_val, int mode)
{
    if (mode & 1) *step_ctr = step;
    if (mode & 2) *n_prev = n_prev_val;
    if (mode & 4) *step_ctr += 1;
}

// a5 + a6, thread-per-marker variant over the sorted markers: u^m(k) = sum U^m W;
// g = u_k - u^m(k); Delta u += s g (R9).
__global__ void __launch_bounds__(128)
k_interp_correct(const unsigned *__restrict__ skey, int n, Geom g, const float4 *__restrict__ U, MarkerSorted m)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int cx, cy, cz;
    key_to_cell(skey[i], g, cx, cy, cz);
    const float4 fs = m.fs[i];
    float wx[4], wy[4], wz[4];
    peskin4(fs.x, wx);
    peskin4(fs.y, wy);
    peskin4(fs.z, wz);
    int xs[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) xs[j] = wrap(cx - 1 + j, g.nx);
    float ux = 0.f, uy = 0.f, uz = 0.f;
#pragma unroll
    for (int jz = 0; jz < 4; ++jz) {
        const int z = wrap(cz - 1 + jz, g.nz);
#pragma unroll
        for (int jy = 0; jy < 4; ++jy) {
            const int y = wrap(cy - 1 + jy, g.ny);
            const float wyz = wy[jy] * wz[jz];
            const float4 *row = U + (size_t)(z * g.ny + y) * g.nx;
#pragma unroll
            for (int jx = 0; jx < 4; ++jx) {
                const float4 v = row[xs[jx]];
                const float w = wx[jx] * wyz;
                ux = fmaf(v.x, w, ux);
                uy = fmaf(v.y, w, uy);
                uz = fmaf(v.z, w, uz);
            }
        }
    }
    const float4 uk = m.uk[i];
    const float gx = uk.x - ux, gy = uk.y - uy, gz = uk.z - uz;
    float4 du = m.du[i];
    du.x = fmaf(fs.w, gx, du.x);
    du.y = fmaf(fs.w, gy, du.y);
    du.z = fmaf(fs.w, gz, du.z);
    m.du[i] = du;                                    // du.w keeps the cell x index
    m.sg[i] = make_float4(fs.w * gx, fs.w * gy, fs.w * gz, du.w);
}

// weight of the cell at offset j (0..3 <-> c-1..c+2) only
__device__ __forceinline__ float peskin1(float f, int j)
{
    const float q = peskin_root(f);
    const float lin = (j < 2) ? (3.0f - 2.0f * f) : (1.0f + 2.0f * f);
    const float sq = (j == 1 || j == 2) ? q : -q;
    return 0.125f * (lin + sq);
}

// a7, plain gather-by-cell (reference variant, slow; kept for cross-checks): one warp per active word, one lane per
// active cell.  The cell visits the 4x4x4 bins whose stencils reach it in a fixed order and, inside
// a bin, the markers in sorted order, so the sum is order-fixed and free of atomics.
//   LAST = false:  U^{m+1}(X) = U^m(X) + sum_k s_k g_k W_k(X)      (R8)
//   LAST = true :  G(X) = sum_k Delta u_k W_k(X)                    (R10, R11)
template <bool LAST>
__global__ void __launch_bounds__(256)
k_spread_gather(const unsigned *__restrict__ skey, int n, Geom g, const int *__restrict__ bin_first,
                const unsigned *__restrict__ amask, const int *__restrict__ words, const int *__restrict__ n_words,
                const float4 *__restrict__ fs, const float4 *__restrict__ val, float4 *__restrict__ field)
{
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    const int nw = *n_words;
    for (int k = warp; k < nw; k += nwarps) {
        const int w = __ldg(words + k);
        const unsigned bits = __ldg(amask + w);
        if (!((bits >> lane) & 1u)) continue;
        const int row = w / g.nxw;
        const int x = (w - row * g.nxw) * 32 + lane;
        const int z = row / g.ny, y = row - z * g.ny;
        float sx = 0.f, sy = 0.f, sz = 0.f;
        // marker cell c = X + 1 - j, j = stencil offset of X inside the marker's block
#pragma unroll 1
        for (int jz = 0; jz < 4; ++jz) {
            int cz = z + 1 - jz;
            if (g.wallz) { if (cz < 0 || cz >= g.nz) continue; } else cz = wrap(cz, g.nz);
#pragma unroll 1
            for (int jy = 0; jy < 4; ++jy) {
                int cy = y + 1 - jy;
                if (g.wally) { if (cy < 0 || cy >= g.ny) continue; } else cy = wrap(cy, g.ny);
#pragma unroll 1
                for (int jx = 0; jx < 4; ++jx) {
                    int cx = x + 1 - jx;
                    if (g.wallx) { if (cx < 0 || cx >= g.nx) continue; } else cx = wrap(cx, g.nx);
                    const unsigned ckey = (unsigned)((cz * g.ny + cy) * g.nx + cx);
                    int i = bin_first[ckey];
                    if (i < 0) continue;
                    for (; i < n && skey[i] == ckey; ++i) {
                        const float4 f = fs[i];
                        const float4 v = val[i];
                        const float wgt = peskin1(f.x, jx) * peskin1(f.y, jy) * peskin1(f.z, jz);
                        sx = fmaf(v.x, wgt, sx);
                        sy = fmaf(v.y, wgt, sy);
                        sz = fmaf(v.z, wgt, sz);
                    }
                }
            }
        }
        const size_t cell = (size_t)row * g.nx + x;
        if (LAST) {
            field[cell] = make_float4(sx, sy, sz, 0.f);
        } else {
            float4 u = field[cell];
            u.x += sx; u.y += sy; u.z += sz;
            field[cell] = u;
        }
    }
}


// ---------------------------------------------------------------------------------------------
// a7, product path: deterministic spreading in two stages, no atomics on the field.
//
// A "chunk" is the stretch of sorted markers that lie in one lattice row (same cy, cz) and in one
// aligned block of CHUNK_W = 8 cells in x.  A marker of source row (cy, cz) reaches the 16 target
// rows (cy-1+jy, cz-1+jz) and, in x, the cells cx-1 .. cx+2, so a chunk of block j touches the
// window X = 8j-1 .. 8j+9 (CHUNK_W + 3 "entries") of each target row: 16 x-profiles
//     sum_k v_k w_y(jy) w_z(jz) w_x(X_e - cx_k + 1),   X_e = 8j - 1 + e,   one per (jy, jz).
// Stage A sweeps every chunk once, in sorted order, and adds its profiles, together with those of
// the other chunks of its TILE (see below), into the tile's footprint.  Stage B lets every active
// cell add up, in fixed order, the footprints that hold it.  All sums have a fixed order, so the
// result is bitwise reproducible.  Chunks are short (<= 8 cells wide) and uniform in cost.

constexpr int CHUNK_W = 8;
constexpr int CHUNK_ENT_MAX = 14;     // widest window: a last block widened to 11 cells (see ChunkGeom)

// Blocks in x: 8 cells each; when nx % 8 is 1..3 the remainder joins the last block (width 9..11), so
// that every block is at least 4 wide and four consecutive cells (periodic or not) meet at most two
// blocks.  ent = widest window = widest block + 3.
struct ChunkGeom {
    int nbx;     // blocks per row
    int ent;     // entries per (chunk, jy, jz) profile (row pitch of T)
};

inline ChunkGeom chunk_geom(int nx)
{
    ChunkGeom c;
    const int rem = nx % CHUNK_W;
    c.nbx = nx / CHUNK_W + ((rem >= 4 || nx < CHUNK_W) ? 1 : 0);
    if (c.nbx < 1) c.nbx = 1;
    const int last_w = nx - (c.nbx - 1) * CHUNK_W;
    c.ent = (last_w > CHUNK_W ? last_w : CHUNK_W) + 3;
    return c;
}

__device__ __forceinline__ int chunk_block(int cx, int nbx) { return min(cx >> 3, nbx - 1); }

// chunk_of[row * nbx + block] packs (chunk id, first entry lo, last entry hi) of the chunk registered there,
// or -1:  id in bits 0..22, lo in bits 23..26, hi in bits 27..30.
constexpr int CHUNK_ID_BITS = 23;
constexpr int CHUNK_ID_MAX = (1 << CHUNK_ID_BITS) - 1;
__device__ __forceinline__ int chunk_pack(int id, int lo, int hi) { return id | (lo << 23) | (hi << 27); }

struct ChunkTable {
    int *first, *end;   // sorted-marker range [first, end) of the chunk
    int *slot;          // index into chunk_of (= row * nbx + block)
};

// a3 (second part): one bit per sorted marker, set where a chunk starts.  Bits at and beyond n are
// set as well, so a forward search for the next chunk start always terminates.
__global__ void __launch_bounds__(256)
k_chunk_heads(const unsigned *__restrict__ skey, int n, Geom g, ChunkGeom cg, unsigned *__restrict__ headbits)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool head = true;
    if (i > 0 && i < n) {
        const unsigned key = skey[i], pk = skey[i - 1];
        const int row = (int)(key / (unsigned)g.nx), prow = (int)(pk / (unsigned)g.nx);
        head = (prow != row) || (chunk_block((int)key - row * g.nx, cg.nbx) != chunk_block((int)pk - prow * g.nx, cg.nbx));
    }
    const unsigned vote = __ballot_sync(0xffffffffu, head);
    if ((threadIdx.x & 31) == 0) headbits[i >> 5] = vote;
}

// set the bits x0..x1 (inclusive, 0 <= x0 <= x1 < nx) of one row of the active-cell mask
__device__ __forceinline__ void mark_span(unsigned *__restrict__ amask, int rowbase, int x0, int x1)
{
    for (int w = x0 >> 5; w <= (x1 >> 5); ++w) {
        const int lo = max(x0 - (w << 5), 0), hi = min(x1 - (w << 5), 31);
        atomicOr(amask + rowbase + w, (0xffffffffu >> (31 - hi)) & (0xffffffffu << lo));
    }
}

// a3: list of the non-zero words of the active-cell mask, in (nearly) ascending order: every warp
// scans a contiguous stretch of the mask 32 words at a time and appends its hits in order.  The
// spatial order is what makes the list-driven passes (moments, collect, stream-collide of the active
// words) touch neighbouring lines one after the other.
__global__ void __launch_bounds__(256)
k_compact_words(const unsigned *__restrict__ amask, int n_mask_words, int *__restrict__ words, int *__restrict__ n_words)
{
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    const int per = ((n_mask_words + nwarps - 1) / nwarps + 31) & ~31;      // words per warp, multiple of 32
    const int beg = warp * per, end = min(beg + per, n_mask_words);
    for (int k0 = beg; k0 < end; k0 += 32) {
        const int k = k0 + lane;
        const bool nz = k < end && amask[k] != 0u;
        const unsigned vote = __ballot_sync(0xffffffffu, nz);
        if (!vote) continue;
        int base = 0;
        if (lane == 0) base = atomicAdd(n_words, __popc(vote));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (nz) words[base + __popc(vote & ((1u << lane) - 1u))] = k;
    }
}

// a3 (third part): the first marker of every chunk finds the chunk's end, takes a chunk id and
// registers the chunk in chunk_of.  Chunks beyond `cap` are dropped and flagged in *status (bit 1).
__global__ void __launch_bounds__(256)
k_chunks(const unsigned *__restrict__ skey, int n, Geom g, ChunkGeom cg, const unsigned *__restrict__ headbits,
         ChunkTable ct, int cap, int *__restrict__ n_chunks, int *__restrict__ n_entries, int *__restrict__ chunk_of,
         int *__restrict__ status)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const unsigned myword = (i < n) ? headbits[i >> 5] : 0u;
    const bool head = (myword >> lane) & 1u;
    int slot = 0, end = 0, lo = 0, hi = 0;
    if (head) {
        // next set bit after i
        int wi = i >> 5;
        unsigned w = (lane == 31) ? 0u : (myword & (0xffffffffu << (lane + 1)));
        while (w == 0u) w = headbits[++wi];
        end = (wi << 5) + __ffs(w) - 1;
        if (end > n) end = n;
        const unsigned key = skey[i], lk = skey[end - 1];
        const int row = (int)(key / (unsigned)g.nx);
        const int cx = (int)key - row * g.nx;
        const int blk = chunk_block(cx, cg.nbx);
        slot = row * cg.nbx + blk;
        lo = cx - blk * CHUNK_W;                                   // window of the first marker starts at entry lo
        hi = ((int)lk - row * g.nx) - blk * CHUNK_W + 3;           // window of the last marker ends at entry hi
    }
    // chunk ids: one atomic per block (warp counts -> block scan), ids ascend with the marker index inside a block
    __shared__ int s_cnt[8], s_ent[8], s_base;
    const int wib = threadIdx.x >> 5;
    const unsigned vote = __ballot_sync(0xffffffffu, head);
    int ne = head ? hi - lo + 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ne += __shfl_xor_sync(0xffffffffu, ne, o);
    if (lane == 0) { s_cnt[wib] = __popc(vote); s_ent[wib] = ne; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int tc = 0, te = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { const int t = s_cnt[w]; s_cnt[w] = tc; tc += t; te += s_ent[w]; }
        s_base = tc ? atomicAdd(n_chunks, tc) : 0;
        if (te) atomicAdd(n_entries, te);
    }
    __syncthreads();
    if (!head) return;
    const int c = s_base + s_cnt[wib] + __popc(vote & ((1u << lane) - 1u));
    if (c >= cap) { atomicOr(status, 2); return; }
    ct.first[c] = i; ct.end[c] = end; ct.slot[c] = slot;
    chunk_of[slot] = chunk_pack(c, lo, hi);
}

// a3 (fourth part): one half-warp per chunk marks the chunk's cells -- the x span cx_first-1 ..
// cx_last+2 in each of the 16 target rows, one row per lane -- in the active-cell bitmask.
__global__ void __launch_bounds__(256)
k_chunk_publish(Geom g, ChunkGeom cg, ChunkTable ct, const int *__restrict__ n_chunks, int cap,
                const int *__restrict__ chunk_of, unsigned *__restrict__ amask)
{
    const int l = threadIdx.x & 15;
    const int hw = (blockIdx.x * blockDim.x + threadIdx.x) >> 4;
    const int nhw = (gridDim.x * blockDim.x) >> 4;
    const int nc = min(*n_chunks, cap);
    for (int c = hw; c < nc; c += nhw) {
        const int slot = ct.slot[c];
        const int packed = chunk_of[slot];
        const int lo = (packed >> 23) & 15, hi = (packed >> 27) & 15;
        const int row = slot / cg.nbx;
        const int blk = slot - row * cg.nbx;
        const int cz = row / g.ny, cy = row - cz * g.ny;
        // x span [xa, xb] = entries lo..hi, entry e <-> X = 8 blk - 1 + e; wrapped on a periodic axis
        const int xa = blk * CHUNK_W - 1 + lo, xb = blk * CHUNK_W - 1 + hi;
        int x0a, x1a, x0b = 0, x1b = -1;
        if (xb - xa + 1 >= g.nx) { x0a = 0; x1a = g.nx - 1; }
        else if (xa < 0) { x0a = xa + g.nx; x1a = g.nx - 1; x0b = 0; x1b = xb; }
        else if (xb >= g.nx) { x0a = xa; x1a = g.nx - 1; x0b = 0; x1b = xb - g.nx; }
        else { x0a = xa; x1a = xb; }
        const int y = wrap(cy - 1 + (l >> 2), g.ny);
        const int z = wrap(cz - 1 + (l & 3), g.nz);
        const int rowbase = (z * g.ny + y) * g.nxw;
        mark_span(amask, rowbase, x0a, x1a);
        if (x1b >= x0b) mark_span(amask, rowbase, x0b, x1b);
    }
}

// a3 (last part): expand the active words into a list of active cell indices (order arbitrary; every
// consumer treats the cells independently).
__global__ void __launch_bounds__(256)
k_active_cells(Geom g, const unsigned *__restrict__ amask, const int *__restrict__ words,
               const int *__restrict__ n_words, int *__restrict__ cells, int *__restrict__ n_cells)
{
    const int lane = threadIdx.x & 31;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const int nw = *n_words;
    for (int k0 = tid - lane; k0 < nw; k0 += stride) {
        const int k = k0 + lane;
        int w = 0;
        unsigned bits = 0u;
        if (k < nw) { w = words[k]; bits = amask[w]; }
        const int cnt = __popc(bits);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        int base = 0;
        if (lane == 0 && total) base = atomicAdd(n_cells, total);
        base = __shfl_sync(0xffffffffu, base, 0) + incl - cnt;
        const int row = w / g.nxw;
        const int cell0 = row * g.nx + (w - row * g.nxw) * 32;
        while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            cells[base++] = cell0 + b;
        }
    }
}

struct Acc3 { float x, y, z; };

// a5 + a6, by chunk (LBM_OPT_INTERP = 3, a measured comparison: north_star's "stage the stencil in shared
// memory"): one warp per chunk (chunks dealt by an atomic cursor).  All stencils of a chunk lie
// in the chunk's window: 16 rows (jy, jz) x (CHUNK_W + 3) cells of U, 2.8 KB.  The warp stages that
// window in shared memory with one round of coalesced loads (two rows per round, a half-warp each) and
// then every lane interpolates one marker of the chunk from shared memory: the 64 gathers of a marker
// are shared-memory reads instead of L1 / L2 round trips.  Measured slower than the lane-per-sorted-marker
// gather (W4 0.38 vs 0.31 ms per step, W4lit 0.18 vs 0.08): a chunk fills 23 of 32 lanes on W4 and 5 on W4lit.
constexpr int ICHUNK_WARPS = 4;

__global__ void __launch_bounds__(ICHUNK_WARPS * 32)
k_interp_chunks(const unsigned *__restrict__ skey, Geom g, ChunkGeom cg, ChunkTable ct, const int *__restrict__ n_chunks,
                int cap, int *__restrict__ cursor, const float4 *__restrict__ U, MarkerSorted m)
{
    __shared__ float4 s_win[ICHUNK_WARPS][16 * CHUNK_ENT_MAX];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = lane & 15, h = lane >> 4;
    const int nc = min(*n_chunks, cap);
    const int ent = cg.ent;
    float4 *win = s_win[warp];
    for (;;) {
        int c = 0;
        if (lane == 0) c = atomicAdd(cursor, 1);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= nc) break;
        const int i0 = __ldg(ct.first + c), i1 = __ldg(ct.end + c), slot = __ldg(ct.slot + c);
        const int row = slot / cg.nbx;
        const int x0 = (slot - row * cg.nbx) * CHUNK_W;
        const int cz = row / g.ny, cy = row - cz * g.ny;
        // stage the window: row r = jz*4 + jy, entry e <-> cell X = x0 - 1 + e (wrapped; out-of-range cells of a
        // wall axis are never used)
        if (l < ent) {
            const int x = wrap(x0 - 1 + l, g.nx);
#pragma unroll
            for (int r2 = 0; r2 < 8; ++r2) {
                const int r = 2 * r2 + h;
                const int y = wrap(cy - 1 + (r & 3), g.ny), z = wrap(cz - 1 + (r >> 2), g.nz);
                win[r * ent + l] = U[(size_t)(z * g.ny + y) * g.nx + x];
            }
        }
        __syncwarp();
        for (int i = i0 + lane; i < i1; i += 32) {
            const unsigned key = skey[i];
            const int ex = (int)(key - (unsigned)row * (unsigned)g.nx) - x0;     // entry of cell cx - 1
            const float4 fs = m.fs[i];
            float wx[4], wy[4], wz[4];
            peskin4(fs.x, wx);
            peskin4(fs.y, wy);
            peskin4(fs.z, wz);
            float ux = 0.f, uy = 0.f, uz = 0.f;
#pragma unroll
            for (int jz = 0; jz < 4; ++jz)
#pragma unroll
                for (int jy = 0; jy < 4; ++jy) {
                    const float wyz = wy[jy] * wz[jz];
                    const float4 *rowp = win + (jz * 4 + jy) * ent + ex;
#pragma unroll
                    for (int jx = 0; jx < 4; ++jx) {
                        const float4 v = rowp[jx];
                        const float w = wx[jx] * wyz;
                        ux = fmaf(v.x, w, ux);
                        uy = fmaf(v.y, w, uy);
                        uz = fmaf(v.z, w, uz);
                    }
                }
            const float4 uk = m.uk[i];
            const float gx = uk.x - ux, gy = uk.y - uy, gz = uk.z - uz;
            float4 du = m.du[i];
            du.x = fmaf(fs.w, gx, du.x);
            du.y = fmaf(fs.w, gy, du.y);
            du.z = fmaf(fs.w, gz, du.z);
            m.du[i] = du;                                // du.w keeps the cell x index
            m.sg[i] = make_float4(fs.w * gx, fs.w * gy, fs.w * gz, du.w);
        }
        __syncwarp();
    }
}

// ---- tiles ---------------------------------------------------------------------------------------
// A "tile" groups the chunks of one x block whose source rows lie in one aligned 4 x 4 block of
// (y, z): up to 16 chunks.  Their 16 x 16 profiles overlap on a footprint of 7 x 7 target rows, so
// one warp sweeps the chunks of a tile one after the other, adds their profiles up in a footprint it
// keeps in shared memory (fixed order) and writes ONE footprint  F[tile][fy][fz][e]  (fy, fz =
// 0..6 <-> target row 4 ty - 1 + fy, 4 tz - 1 + fz; e as in the chunk window).  Stage B then reads
// about 4 footprints per cell instead of 22 profiles, and the profile traffic shrinks ~7x.
//
// tile_mask[tile slot] = x entries (bits 0..13) | y rows (bits 14..20) | z rows (bits 21..27) that
// some chunk of the tile reaches; a footprint element is valid iff its three bits are set (a
// superset of the cells actually reached; the rest is written as zeros).
constexpr int TILE_R = 4;                  // source rows per tile in y and in z (large marker sets; the round-1 sweep)
constexpr int TILE_F = TILE_R + 3;         // footprint rows per tile in y and in z
constexpr int TILE_R_MAX = 4;

// The tile edge is a property of the marker set (tr = 4, 2 or 1 source rows in y and in z): small sets use
// tiles of a single source row so that a few thousand markers still make enough tiles for all SMs.
struct TileGeom {
    int nty, ntz;        // tiles in y and z
    int tr;              // source rows per tile in y and in z
};
inline TileGeom tile_geom(int ny, int nz, int tr = TILE_R)
{
    TileGeom t;
    t.tr = tr;
    t.nty = (ny + tr - 1) / tr;
    t.ntz = (nz + tr - 1) / tr;
    return t;
}

struct TileTable {
    unsigned *mask;      // [tile slots] dense, 0 = no tile
    int *id;             // [tile slots] dense: footprint index of the tile (valid where mask != 0)
    int *slot;           // [tile ids] -> tile slot
    int2 *rec;           // [tile ids][tr*tr]: sorted-marker range [first, end) of the chunk in source row sy + tr sz, (0,0) = none
    // the same records in processing order (longest tile first), so that a warp that draws position k from the work
    // cursor finds everything about its tile with one round of loads
    int4 *ohdr;          // [position] (tile slot, reach mask, tile id, markers of the tile)
    int2 *orec;          // [position][tr*tr] as rec
};

__device__ __forceinline__ int tile_slot_of(int blk, int ty, int tz, const ChunkGeom &cg, const TileGeom &tg)
{
    return (tz * tg.nty + ty) * cg.nbx + blk;
}

// a3: register every chunk in its tile (bits it reaches); the chunk that finds the mask empty
// allocates the tile's footprint index.  One thread per chunk.
__global__ void __launch_bounds__(256)
k_tiles(Geom g, ChunkGeom cg, TileGeom tg, ChunkTable ct, const int *__restrict__ n_chunks, int cap,
        const int *__restrict__ chunk_of, TileTable tt, int tile_cap, int *__restrict__ n_tiles, int *__restrict__ ovf_slot,
        int ovf_cap, int *__restrict__ n_ovf, int *__restrict__ status)
{
    const int nc = min(*n_chunks, cap);
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        const int slot = ct.slot[c];
        const int packed = chunk_of[slot];
        const int lo = (packed >> 23) & 15, hi = (packed >> 27) & 15;
        const int row = slot / cg.nbx;
        const int blk = slot - row * cg.nbx;
        const int cz = row / g.ny, cy = row - cz * g.ny;
        const unsigned xbits = ((1u << (hi - lo + 1)) - 1u) << lo;
        const unsigned ybits = 0xFu << (cy % tg.tr), zbits = 0xFu << (cz % tg.tr);
        const int ts = tile_slot_of(blk, cy / tg.tr, cz / tg.tr, cg, tg);
        const unsigned old = atomicOr(tt.mask + ts, xbits | (ybits << 14) | (zbits << 21));
        if (old == 0u) {
            const int id = atomicAdd(n_tiles, 1);
            if (id < tile_cap) {
                tt.slot[id] = ts; tt.id[ts] = id;
                int2 *z = tt.rec + (size_t)id * (tg.tr * tg.tr);
                for (int i = 0; i < tg.tr * tg.tr; ++i) z[i] = make_int2(0, 0);
            } else {
                // no footprint left: undo the registration so that the slot is not stuck with a stale mask once a
                // later step fits again (chunks that find the slot non-empty below re-register into id = -1 and are
                // dropped for this step only; k_clear_prev clears the slots listed in ovf_slot)
                tt.id[ts] = -1;
                const int o = atomicAdd(n_ovf, 1);
                if (o < ovf_cap) ovf_slot[o] = ts;
                atomicOr(status, 2);
            }
        }
    }
}

// a3: every chunk writes its marker range into the record of its tile (after k_tiles has handed out the ids).
__global__ void __launch_bounds__(256)
k_tile_fill(Geom g, ChunkGeom cg, TileGeom tg, ChunkTable ct, const int *__restrict__ n_chunks, int cap, TileTable tt)
{
    const int nc = min(*n_chunks, cap);
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        const int slot = ct.slot[c];
        const int row = slot / cg.nbx;
        const int blk = slot - row * cg.nbx;
        const int cz = row / g.ny, cy = row - cz * g.ny;
        const int id = tt.id[tile_slot_of(blk, cy / tg.tr, cz / tg.tr, cg, tg)];
        if (id >= 0) tt.rec[(size_t)id * (tg.tr * tg.tr) + (cy % tg.tr) + tg.tr * (cz % tg.tr)] = make_int2(ct.first[c], ct.end[c]);
    }
}

// a3: order the tiles by decreasing marker count (8 size classes: >= 1024, >= 512, ... , < 16), so that the
// sweep, which hands tiles out through a cursor, starts the long ones first and ends on short ones
// (longest-processing-time-first; the order inside a class is arbitrary).  Two passes: count per
// class, then place.  bucket[0..7] = class counts, bucket[8..15] = fill cursors.
__device__ __forceinline__ int tile_size_class(const int2 *__restrict__ rec, int nr)
{
    int n = 0;
    for (int r = 0; r < nr; ++r) { const int2 v = __ldg(rec + r); n += v.y - v.x; }
    const int c = 27 - __clz(max(n, 1));       // floor(log2 n) - 4
    return 7 - min(max(c, 0), 7);              // class 0 = largest
}

__global__ void __launch_bounds__(256)
k_tile_count(TileTable tt, int nr, const int *__restrict__ n_tiles, int tile_cap, int *__restrict__ bucket)
{
    const int nt = min(*n_tiles, tile_cap);
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < nt; t += gridDim.x * blockDim.x)
        atomicAdd(bucket + tile_size_class(tt.rec + (size_t)t * nr, nr), 1);
}

__global__ void __launch_bounds__(256)
k_tile_place(TileTable tt, int nr, const int *__restrict__ n_tiles, int tile_cap, int *__restrict__ bucket, int *__restrict__ order)
{
    const int nt = min(*n_tiles, tile_cap);
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < nt; t += gridDim.x * blockDim.x) {
        const int c = tile_size_class(tt.rec + (size_t)t * nr, nr);
        int base = 0;
        for (int q = 0; q < c; ++q) base += bucket[q];
        const int pos = base + atomicAdd(bucket + 8 + c, 1);
        order[pos] = t;
        int n = 0;
        for (int r = 0; r < nr; ++r) { const int2 v = tt.rec[(size_t)t * nr + r]; tt.orec[(size_t)pos * nr + r] = v; n += v.y - v.x; }
        const int ts = tt.slot[t];
        tt.ohdr[pos] = make_int4(ts, (int)tt.mask[ts], t, n);
    }
}

// ---- asynchronous bulk copies global -> shared (TMA, 1-D) completing on an mbarrier ---------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// Stage A: one WARP per tile, no block-level synchronisation at all.  The warp walks through the
// source rows of its tile that hold a chunk, in ascending order, and sweeps each chunk with
// lane = h*16 + l: l = jy*4 + jz is the target-row offset whose profile the lane accumulates, h the
// half of the 4-cell x window it owns (h = 0: the two left cells, h = 1: the two right cells), both
// in registers.  When the sweep moves on to the next cell the leftmost window cell is final: the
// lane adds it to the tile's footprint, which the warp keeps in shared memory (the 16 lanes of a
// chunk hit 16 different footprint rows, and chunks follow one another, so there is no conflict and
// the order of every sum is fixed), and the window shifts by one (the cell that crosses from the
// right half to the left half travels by shuffle).  Control flow is uniform across the warp.
//
// The marker data of a chunk (value, x weights, y-z weights: three contiguous ranges of the sorted
// arrays) comes through the warp's own shared-memory buffers by asynchronous bulk copies (TMA),
// SPREAD_PIECE markers at a time through a ring of SPREAD_STAGES buffers that runs ACROSS chunks, so
// the sweep never waits on a global load per marker.  Tiles are handed out, longest first, through an
// atomic cursor.
//
// Shared memory (dynamic), per warp: footprint [7*7][ent][3] floats, then STAGES x { val[PIECE] float4,
// wx[PIECE] float4, wyz[PIECE][16] float }.
#ifndef TILE_WARPS_CFG
#define TILE_WARPS_CFG 4
#define TILE_MINB_CFG 5
#define SPREAD_PIECE_CFG 16
#define SPREAD_STAGES_CFG 2
#endif
constexpr int TILE_WARPS = TILE_WARPS_CFG;
constexpr int SPREAD_PIECE = SPREAD_PIECE_CFG;
constexpr int SPREAD_STAGES = SPREAD_STAGES_CFG;     // ring of staging buffers per warp: STAGES - 1 pieces in flight
constexpr int SPREAD_PIECE_BYTES = SPREAD_PIECE * 96;

inline size_t spread_warp_smem(const ChunkGeom &cg)
{
    const size_t foot = ((size_t)TILE_F * TILE_F * (size_t)cg.ent * 3 * sizeof(float) + 127) / 128 * 128;
    return foot + SPREAD_STAGES * SPREAD_PIECE_BYTES;
}
inline size_t spread_tiles_smem(const ChunkGeom &cg) { return (size_t)TILE_WARPS * spread_warp_smem(cg); }

__global__ void __launch_bounds__(TILE_WARPS * 32, TILE_MINB_CFG)
k_spread_tiles(ChunkGeom cg, const int2 *__restrict__ tile_rec, const int *__restrict__ tile_slot,
               const unsigned *__restrict__ tile_mask, const int *__restrict__ n_tiles, int tile_cap,
               int *__restrict__ cursor, const int *__restrict__ order, const float4 *__restrict__ wx4,
               const float *__restrict__ wyz16, const float4 *__restrict__ val, const int *__restrict__ fdst,
               float4 *__restrict__ F, int warp_smem)
{
    extern __shared__ __align__(128) char smem[];
    __shared__ unsigned long long s_bar[TILE_WARPS][SPREAD_STAGES];
    __shared__ int s_n[TILE_WARPS][SPREAD_STAGES];     // markers in the piece a stage holds
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = lane & 15, h = lane >> 4;
    const int nt = min(*n_tiles, tile_cap);
    const int ent = cg.ent;
    float *foot = reinterpret_cast<float *>(smem + (size_t)warp * warp_smem);
    char *stage = smem + (size_t)warp * warp_smem + (warp_smem - SPREAD_STAGES * SPREAD_PIECE_BYTES);
    unsigned long long *bar = s_bar[warp];
    if (lane < SPREAD_STAGES) mbar_init(&bar[lane], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncwarp();
    unsigned phase = 0u;                                 // bit b: parity the next wait on bar[b] uses
    const int nfoot = TILE_F * TILE_F * ent;             // footprint elements
    const int jy = l >> 2, jz = l & 3;
    for (;;) {
        int t = 0;
        if (lane == 0) { t = atomicAdd(cursor, 1); t = t < nt ? __ldg(order + t) : nt; }
        t = __shfl_sync(0xffffffffu, t, 0);
        if (t >= nt) break;
        // lane r < 16: sorted-marker range of the chunk in source row r = sy + 4 sz ((0,0) = none)
        const int2 rec = __ldg(tile_rec + (size_t)t * 16 + l);
        const unsigned present = __ballot_sync(0xffffffffu, rec.y > rec.x) & 0xffffu;
        const int ts = __ldg(tile_slot + t);
        const int x0 = (ts % cg.nbx) * CHUNK_W;
        // piece stream over the chunks of the tile: (row, offset) of the next piece to issue
        unsigned irest = present;
        int ioff = 0;
        int n_issued = 0;
        auto issue = [&]() {                             // next piece of the stream into stage n_issued % STAGES
            if (!irest) return;
            const int b = n_issued % SPREAD_STAGES;
            const int r = __ffs(irest) - 1;
            const int first = __shfl_sync(0xffffffffu, rec.x, r), end = __shfl_sync(0xffffffffu, rec.y, r);
            const int j0 = first + ioff;
            const int n = min(SPREAD_PIECE, end - j0);
            if (lane == 0) {
                char *dst = stage + b * SPREAD_PIECE_BYTES;
                s_n[warp][b] = n;
                mbar_expect_tx(&bar[b], (unsigned)n * 96u);
                bulk_g2s(dst, val + j0, (unsigned)n * 16u, &bar[b]);
                bulk_g2s(dst + SPREAD_PIECE * 16, wx4 + j0, (unsigned)n * 16u, &bar[b]);
                bulk_g2s(dst + SPREAD_PIECE * 32, wyz16 + (size_t)j0 * 16, (unsigned)n * 64u, &bar[b]);
            }
            ioff += n;
            if (j0 + n == end) { irest &= irest - 1; ioff = 0; }
            ++n_issued;
        };
#pragma unroll
        for (int i = 0; i < SPREAD_STAGES - 1; ++i) issue();
        // zero the footprint while the first piece is in flight
        for (int i = lane; i < (nfoot * 3 + 3) / 4; i += 32) reinterpret_cast<float4 *>(foot)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncwarp();
        // consumer state: row being swept and how many of its markers are still to come
        unsigned crest = present;
        int cleft = 0;
        float *frow = foot;
        Acc3 p{0.f, 0.f, 0.f}, q{0.f, 0.f, 0.f};         // window cells (e + 2h, e + 2h + 1)
        int e = 0;
        for (int k = 0; k < n_issued; ++k) {
            issue();                                     // into the stage the previous round released (__syncwarp below)
            const int b = k % SPREAD_STAGES;
            mbar_wait(&bar[b], (phase >> b) & 1u);
            phase ^= 1u << b;
            const int n_cur = s_n[warp][b];
            const char *src = stage + b * SPREAD_PIECE_BYTES;
            const float4 *sv = reinterpret_cast<const float4 *>(src);
            const float2 *sw = reinterpret_cast<const float2 *>(src + SPREAD_PIECE * 16) + h;
            const float *sz = reinterpret_cast<const float *>(src + SPREAD_PIECE * 32) + l;
            if (cleft == 0) {                            // this piece starts a new source row
                const int r = __ffs(crest) - 1;
                crest &= crest - 1;
                cleft = __shfl_sync(0xffffffffu, rec.y - rec.x, r);
                frow = foot + (((r & 3) + jy) * TILE_F + ((r >> 2) + jz)) * ent * 3;
                p = Acc3{0.f, 0.f, 0.f}; q = Acc3{0.f, 0.f, 0.f};
                e = __float_as_int(sv[0].w) - x0;        // window start = entry of the first marker's cx - 1
            }
            auto flush = [&](int ee, const Acc3 &a) {
                float *d = frow + ee * 3;
                d[0] += a.x; d[1] += a.y; d[2] += a.z;
            };
#pragma unroll 4
            for (int j = 0; j < n_cur; ++j) {
                const float4 v = sv[j];
                const float2 w = sw[2 * j];
                const float wz = sz[16 * j];
                const int em = __float_as_int(v.w) - x0;
                if (em != e) {                           // warp-uniform: the sweep moves on to another cell
#pragma unroll 1
                    do {                                 // the leftmost window cell is complete
                        if (h == 0) flush(e, p);
                        const float tx = __shfl_down_sync(0xffffffffu, p.x, 16);
                        const float ty = __shfl_down_sync(0xffffffffu, p.y, 16);
                        const float tz = __shfl_down_sync(0xffffffffu, p.z, 16);
                        p = q;
                        q.x = h ? 0.f : tx; q.y = h ? 0.f : ty; q.z = h ? 0.f : tz;
                    } while (++e < em);
                }
                const float vx = v.x * wz, vy = v.y * wz, vz = v.z * wz;
                p.x = fmaf(w.x, vx, p.x); p.y = fmaf(w.x, vy, p.y); p.z = fmaf(w.x, vz, p.z);
                q.x = fmaf(w.y, vx, q.x); q.y = fmaf(w.y, vy, q.y); q.z = fmaf(w.y, vz, q.z);
            }
            cleft -= n_cur;
            if (cleft == 0) {                            // the row's last window: entries e .. e+3 (= hi)
                flush(e + 2 * h, p);
                flush(e + 2 * h + 1, q);
            }
            __syncwarp();                                // every lane is done with stage b (and with the footprint row)
        }
        // hand the footprint elements some chunk of the tile can reach (mask product) to the cells that consume
        // them (collect plan fdst, mdf_kernels.cuh); the rest is never read
        const unsigned m = __ldg(tile_mask + ts);
        const int *__restrict__ dst = fdst + (size_t)t * nfoot;
        for (int idx = lane; idx < nfoot; idx += 32) {
            const int fyz = idx / ent, ee = idx - fyz * ent;
            const int fy = fyz / TILE_F, fz = fyz - fy * TILE_F;
            if ((m >> ee) & (m >> (14 + fy)) & (m >> (21 + fz)) & 1u) {
                const int o = __ldg(dst + idx);
                const float *s = foot + idx * 3;
                if (o >= 0) F[o] = make_float4(s[0], s[1], s[2], 0.f);
            }
        }
        __syncwarp();
    }
}

// a7, atomic variant (the paper's ib_force2 idea, kept as a measured comparison):
// every marker adds its 64 contributions with global float atomics.  Not deterministic.
__global__ void __launch_bounds__(128)
k_spread_atomic(const unsigned *__restrict__ skey, int n, Geom g, const float4 *__restrict__ fs,
                const float4 *__restrict__ val, float4 *__restrict__ field)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int cx, cy, cz;
    key_to_cell(skey[i], g, cx, cy, cz);
    const float4 f = fs[i];
    const float4 v = val[i];
    float wx[4], wy[4], wz[4];
    peskin4(f.x, wx);
    peskin4(f.y, wy);
    peskin4(f.z, wz);
#pragma unroll 1
    for (int jz = 0; jz < 4; ++jz) {
        const int z = wrap(cz - 1 + jz, g.nz);
#pragma unroll 1
        for (int jy = 0; jy < 4; ++jy) {
            const int y = wrap(cy - 1 + jy, g.ny);
            const float wyz = wy[jy] * wz[jz];
            float *row = reinterpret_cast<float *>(field + (size_t)(z * g.ny + y) * g.nx);
#pragma unroll
            for (int jx = 0; jx < 4; ++jx) {
                const int x = wrap(cx - 1 + jx, g.nx);
                const float w = wx[jx] * wyz;
                atomicAdd(row + 4 * x + 0, v.x * w);
                atomicAdd(row + 4 * x + 1, v.y * w);
                atomicAdd(row + 4 * x + 2, v.z * w);
            }
        }
    }
}

// zero G on the active cells (needed before the atomic variant accumulates into it)
__global__ void __launch_bounds__(256)
k_zero_active(Geom g, const unsigned *__restrict__ amask, const int *__restrict__ words,
              const int *__restrict__ n_words, float4 *__restrict__ field)
{
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    const int nw = *n_words;
    for (int k = warp; k < nw; k += nwarps) {
        const int w = words[k];
        if (!((amask[w] >> lane) & 1u)) continue;
        const int row = w / g.nxw;
        const int x = (w - row * g.nxw) * 32 + lane;
        field[(size_t)row * g.nx + x] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// read-back helpers: scatter sorted per-marker data to the caller's original order
__global__ void __launch_bounds__(256)
k_read_markers(const unsigned *__restrict__ skey, const int *__restrict__ perm, int n, Geom g,
               const float4 *__restrict__ fs, const float4 *__restrict__ du, float *__restrict__ pos,
               float *__restrict__ force, int *__restrict__ cell)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int k = perm[i];
    const unsigned key = skey[i];
    if (pos) {
        int cx, cy, cz;
        key_to_cell(key, g, cx, cy, cz);
        const float4 f = fs[i];
        pos[3 * k + 0] = (float)cx + f.x;
        pos[3 * k + 1] = (float)cy + f.y;
        pos[3 * k + 2] = (float)cz + f.z;
    }
    if (force) {
        const float4 d = du[i];
        force[3 * k + 0] = d.x; force[3 * k + 1] = d.y; force[3 * k + 2] = d.z;
    }
    if (cell) cell[k] = (int)key;
}

// =================================================================================================
// The paper's own kernel designs, kept as measured comparisons; none of them
// is on the default path.  They produce the same fields as the product kernels (U bit-identical,
// atomics up to summation order).

// general Peskin 4-point kernel w(r) (R6), used where the stencil offset is not known at compile time
__device__ __forceinline__ float peskin_w(float r)
{
    const float a = fabsf(r);
    if (a >= 2.0f) return 0.0f;
    if (a <= 1.0f) return 0.125f * (3.0f - 2.0f * a + sqrtf(fmaf(4.0f * a, 1.0f - a, 1.0f)));
    return 0.125f * (5.0f - 2.0f * a - sqrtf(fmaf(-4.0f * a, a, fmaf(12.0f, a, -7.0f))));
}

// inverse of the sort permutation: inv[original index] = sorted index
__global__ void __launch_bounds__(256)
k_invert_perm(const int *__restrict__ perm, int n, int *__restrict__ inv)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) inv[perm[i]] = i;
}

// f4, ib_force1 as the paper has it (Alg.1): one thread per Lagrangian point in the
// CALLER's order, no reordering, so neighbouring threads gather from unrelated places (P:152
// "memory accesses are often not coalesced").  Same arithmetic as k_interp_correct.
__global__ void __launch_bounds__(128)
k_interp_caller_order(const unsigned *__restrict__ skey, const int *__restrict__ inv, int n, Geom g,
                      const float4 *__restrict__ U, MarkerSorted m)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int i = inv[k];
    int cx, cy, cz;
    key_to_cell(skey[i], g, cx, cy, cz);
    const float4 fs = m.fs[i];
    float wx[4], wy[4], wz[4];
    peskin4(fs.x, wx);
    peskin4(fs.y, wy);
    peskin4(fs.z, wz);
    float ux = 0.f, uy = 0.f, uz = 0.f;
#pragma unroll
    for (int jz = 0; jz < 4; ++jz) {
        const int z = wrap(cz - 1 + jz, g.nz);
#pragma unroll
        for (int jy = 0; jy < 4; ++jy) {
            const int y = wrap(cy - 1 + jy, g.ny);
            const float wyz = wy[jy] * wz[jz];
            const float4 *row = U + (size_t)(z * g.ny + y) * g.nx;
#pragma unroll
            for (int jx = 0; jx < 4; ++jx) {
                const float4 v = row[wrap(cx - 1 + jx, g.nx)];
                const float w = wx[jx] * wyz;
                ux = fmaf(v.x, w, ux);
                uy = fmaf(v.y, w, uy);
                uz = fmaf(v.z, w, uz);
            }
        }
    }
    const float4 uk = m.uk[i];
    const float gx = uk.x - ux, gy = uk.y - uy, gz = uk.z - uz;
    float4 du = m.du[i];
    du.x = fmaf(fs.w, gx, du.x);
    du.y = fmaf(fs.w, gy, du.y);
    du.z = fmaf(fs.w, gz, du.z);
    m.du[i] = du;
    m.sg[i] = make_float4(fs.w * gx, fs.w * gy, fs.w * gz, du.w);
}

// The warp-cooperative interpolation north_star names, kept as a measured comparison
// (LBM_OPT_INTERP = 2): one warp per sorted marker, lane = (jz half, jy, jx): every lane loads two
// of the 64 stencil cells (the x-quads of a warp-load are 64 contiguous bytes), weighs them, and the
// warp reduces the three components with shuffles.  36 warp instructions per marker against 25 per
// marker (800 per 32 markers) for the lane-per-marker gather, and 1/32 of the loads in flight per warp.
__global__ void __launch_bounds__(256)
k_interp_warp_per_marker(const unsigned *__restrict__ skey, int n, Geom g, const float4 *__restrict__ U, MarkerSorted m)
{
    const int lane = threadIdx.x & 31;
    const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (i >= n) return;
    int cx, cy, cz;
    key_to_cell(skey[i], g, cx, cy, cz);
    const float4 fs = m.fs[i];
    const int jx = lane & 3, jy = (lane >> 2) & 3, jzh = lane >> 4;
    const float wxy = peskin1(fs.x, jx) * peskin1(fs.y, jy);
    const int x = wrap(cx - 1 + jx, g.nx), y = wrap(cy - 1 + jy, g.ny);
    float ux = 0.f, uy = 0.f, uz = 0.f;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int jz = 2 * jzh + q;
        const int z = wrap(cz - 1 + jz, g.nz);
        const float4 v = U[(size_t)(z * g.ny + y) * g.nx + x];
        const float w = wxy * peskin1(fs.z, jz);
        ux = fmaf(v.x, w, ux); uy = fmaf(v.y, w, uy); uz = fmaf(v.z, w, uz);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ux += __shfl_xor_sync(0xffffffffu, ux, o);
        uy += __shfl_xor_sync(0xffffffffu, uy, o);
        uz += __shfl_xor_sync(0xffffffffu, uz, o);
    }
    if (lane != 0) return;
    const float4 uk = m.uk[i];
    const float gx = uk.x - ux, gy = uk.y - uy, gz = uk.z - uz;
    float4 du = m.du[i];
    du.x = fmaf(fs.w, gx, du.x);
    du.y = fmaf(fs.w, gy, du.y);
    du.z = fmaf(fs.w, gz, du.z);
    m.du[i] = du;
    m.sg[i] = make_float4(fs.w * gx, fs.w * gy, fs.w * gz, du.w);
}

// f4, ib_force2 as the paper has it (Alg.2): one CUDA block of 5 x 5 x 5 threads per
// Lagrangian point, thread (a,b,c) adds the contribution to the cell round(x) + (a,b,c) - 2 with
// atomicAdd.  At most 4 of the 5 weights per axis are non-zero (R7).
__global__ void __launch_bounds__(125)
k_spread_block125(const unsigned *__restrict__ skey, int n, Geom g, const float4 *__restrict__ fs,
                  const float4 *__restrict__ val, float4 *__restrict__ field)
{
    const int i = blockIdx.x;
    if (i >= n) return;
    int cx, cy, cz;
    key_to_cell(skey[i], g, cx, cy, cz);
    const float4 f = fs[i];
    const float4 v = val[i];
    const int a = threadIdx.x % 5, b = (threadIdx.x / 5) % 5, c = threadIdx.x / 25;
    // nearest cell round(x) = cell + (fraction >= 1/2); distance of the point to the thread's cell
    const int rx = f.x >= 0.5f ? 1 : 0, ry = f.y >= 0.5f ? 1 : 0, rz = f.z >= 0.5f ? 1 : 0;
    const int ox = rx + a - 2, oy = ry + b - 2, oz = rz + c - 2;
    const float w = peskin_w(f.x - (float)ox) * peskin_w(f.y - (float)oy) * peskin_w(f.z - (float)oz);
    if (w == 0.0f) return;
    const int x = wrap(cx + ox, g.nx), y = wrap(cy + oy, g.ny), z = wrap(cz + oz, g.nz);
    float *dst = reinterpret_cast<float *>(field + (size_t)(z * g.ny + y) * g.nx + x);
    atomicAdd(dst + 0, v.x * w);
    atomicAdd(dst + 1, v.y * w);
    atomicAdd(dst + 2, v.z * w);
}

// f2, lbm_u_start "kernel strategy" as the paper has it: one CUDA block per Lagrangian
// point computes U on the point's 4 x 4 x 4 neighbourhood; the same U(X) is computed by every
// point whose neighbourhood holds X.
__global__ void __launch_bounds__(64)
k_moments_per_marker(const float *__restrict__ src, const __grid_constant__ Geom g, const unsigned *__restrict__ skey,
                     int n, float4 *__restrict__ U)
{
    const int i = blockIdx.x;
    if (i >= n) return;
    int cx, cy, cz;
    key_to_cell(skey[i], g, cx, cy, cz);
    const int x = wrap(cx - 1 + (threadIdx.x & 3), g.nx);
    const int y = wrap(cy - 1 + ((threadIdx.x >> 2) & 3), g.ny);
    const int z = wrap(cz - 1 + (threadIdx.x >> 4), g.nz);
    const Nbr nb = neighbours(g, x, y, z);
    float df[NQ], drho, ux, uy, uz;
    pull_cell(src, g, nb, x, y, z, df);
    moments(df, drho, ux, uy, uz);
    U[(size_t)(z * g.ny + y) * g.nx + x] = make_float4(ux, uy, uz, 1.0f + drho);
}

// f2, lbm_u_start "box strategy": U on the bounding box of every body.  The paper
// transforms the rest-pose box; here the box is taken from the cells the body's markers occupy in
// this step (tighter), widened by the stencil.  Boxes are kept unwrapped (they may straddle a
// periodic face); box[b] = {xlo, ylo, zlo, xhi, yhi, zhi}.
__global__ void __launch_bounds__(256)
k_body_boxes(MarkerIn m, const BodyDef *__restrict__ defs, const BodyStep *__restrict__ tabs, int *__restrict__ box)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m.n) return;
    const int b = m.body[k];
    const BodyDef d = defs[b];
    const BodyStep t = tabs[b];
    const float4 q4 = __ldg(m.qs + k);
    const float qx = q4.x, qy = q4.y, qz = q4.z;
    const float dx = fmaf(t.R[0], qx, fmaf(t.R[1], qy, fmaf(t.R[2], qz, d.cf[0])));
    const float dy = fmaf(t.R[3], qx, fmaf(t.R[4], qy, fmaf(t.R[5], qz, d.cf[1])));
    const float dz = fmaf(t.R[6], qx, fmaf(t.R[7], qy, fmaf(t.R[8], qz, d.cf[2])));
    const int cx = d.ci[0] + (int)floorf(dx), cy = d.ci[1] + (int)floorf(dy), cz = d.ci[2] + (int)floorf(dz);
    int *bx = box + 6 * b;
    atomicMin(bx + 0, cx - 1); atomicMin(bx + 1, cy - 1); atomicMin(bx + 2, cz - 1);
    atomicMax(bx + 3, cx + 3); atomicMax(bx + 4, cy + 3); atomicMax(bx + 5, cz + 3);   // + 3: rounding of d - floor(d) (place_axis)
}

__global__ void k_reset_boxes(int *__restrict__ box, int nbodies)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbodies) return;
    for (int a = 0; a < 3; ++a) { box[6 * b + a] = 0x7fffffff; box[6 * b + 3 + a] = -0x7fffffff; }
}

// grid (blocks per body, bodies): the blocks of a body stride over the cells of its box
__global__ void __launch_bounds__(256)
k_moments_box(const float *__restrict__ src, const __grid_constant__ Geom g, const int *__restrict__ box,
              float4 *__restrict__ U)
{
    const int *bx = box + 6 * blockIdx.y;
    const int x0 = bx[0], y0 = bx[1], z0 = bx[2];
    const int ex = min(bx[3] - x0 + 1, g.nx), ey = min(bx[4] - y0 + 1, g.ny), ez = min(bx[5] - z0 + 1, g.nz);
    if (ex <= 0 || ey <= 0 || ez <= 0) return;
    const long long total = (long long)ex * ey * ez;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < total; c += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(c % ex), iy = (int)((c / ex) % ey), iz = (int)(c / ((long long)ex * ey));
        int x = (x0 + ix) % g.nx, y = (y0 + iy) % g.ny, z = (z0 + iz) % g.nz;
        if (x < 0) x += g.nx;
        if (y < 0) y += g.ny;
        if (z < 0) z += g.nz;
        const Nbr nb = neighbours(g, x, y, z);
        float df[NQ], drho, ux, uy, uz;
        pull_cell(src, g, nb, x, y, z, df);
        moments(df, drho, ux, uy, uz);
        U[(size_t)(z * g.ny + y) * g.nx + x] = make_float4(ux, uy, uz, 1.0f + drho);
    }
}

}  // namespace lbmk
