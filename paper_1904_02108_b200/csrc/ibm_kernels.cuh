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

struct MarkerIn {                  // original (caller) order, SoA
    const float *qx, *qy, *qz;     // rest position relative to the body centre, p_k - c (fp64 -> fp32)
    const float *vx, *vy, *vz;     // extra velocity vel_k (R14)
    const float *s;                // area s(k)
    const int *body;
    int n;
};

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
              unsigned *__restrict__ keys, int *__restrict__ status)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m.n) return;
    const int b = m.body[k];
    const Placed p = place_marker(defs[b], tabs[b], m.qx[k], m.qy[k], m.qz[k], g);
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
    float4 *wx;     // the four x weights w(x_k - X), X = cx-1 .. cx+2
    float *wyz;     // [16] per marker: w_y(jy) w_z(jz) at index jy*4+jz
                    // sg.w and du.w carry the marker's cell x index (int bits) for the run sweep
    float4 *uk;     // prescribed velocity u_k, w unused
    float4 *sg;     // s * g^m(k)   (what the U update spreads, P:98 + R8)
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
    const int b = m.body[k];
    const BodyStep t = tabs[b];
    const float qx = m.qx[k], qy = m.qy[k], qz = m.qz[k];
    const Placed p = place_marker(defs[b], t, qx, qy, qz, g);
    out.fs[i] = make_float4(p.fx, p.fy, p.fz, m.s[k]);

    const float ux = fmaf(t.dR[0], qx, fmaf(t.dR[1], qy, fmaf(t.dR[2], qz, m.vx[k])));
    const float uy = fmaf(t.dR[3], qx, fmaf(t.dR[4], qy, fmaf(t.dR[5], qz, m.vy[k])));
    const float uz = fmaf(t.dR[6], qx, fmaf(t.dR[7], qy, fmaf(t.dR[8], qz, m.vz[k])));
    out.uk[i] = make_float4(ux, uy, uz, 0.f);
    out.du[i] = make_float4(0.f, 0.f, 0.f, __int_as_float(p.cx));
    out.sg[i] = make_float4(0.f, 0.f, 0.f, __int_as_float(p.cx));
    // per-step weight tables of the run sweep (the position does not change during the MDF loop)
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
// the active-cell bitmask (one bit per cell, 32 consecutive x per word).  The thread whose
// atomicOr turns a word from 0 to non-zero appends it to the active-word list (warp-aggregated).
__global__ void __launch_bounds__(256)
k_bins(const unsigned *__restrict__ skey, int n, Geom g, int *__restrict__ bin_first, unsigned *__restrict__ amask,
       int *__restrict__ words, int *__restrict__ n_words)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
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
    // the four x cells cx-1..cx+2 fall into at most two words (two runs when they wrap)
#pragma unroll 1
    for (int r = 0; r < 16; ++r) {
        const int y = wrap(cy - 1 + (r & 3), g.ny);
        const int z = wrap(cz - 1 + (r >> 2), g.nz);
        const int rowbase = (z * g.ny + y) * g.nxw;
        int w0 = -1, w1 = -1;
        unsigned b0 = 0, b1 = 0;
        if (head) {
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int x = wrap(cx - 1 + j, g.nx);
                const int w = rowbase + (x >> 5);
                const unsigned bit = 1u << (x & 31);
                if (w0 < 0 || w == w0) { w0 = w; b0 |= bit; }
                else { w1 = w; b1 |= bit; }
            }
        }
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const int w = half ? w1 : w0;
            const unsigned b = half ? b1 : b0;
            bool fresh = false;
            if (w >= 0) fresh = (atomicOr(amask + w, b) == 0u);
            const unsigned vote = __ballot_sync(0xffffffffu, fresh);
            if (vote) {
                int base = 0;
                const int leader = __ffs(vote) - 1;
                if (lane == leader) base = atomicAdd(n_words, __popc(vote));
                base = __shfl_sync(0xffffffffu, base, leader);
                if (fresh) words[base + __popc(vote & ((1u << lane) - 1u))] = w;
            }
        }
    }
}

// Undo what k_bins of the previous step left behind (bitmask words and cell -> first-marker
// entries), so neither needs a full-lattice memset per step.
__global__ void __launch_bounds__(256)
k_clear_prev(const unsigned *__restrict__ skey_prev, const int *__restrict__ n_prev, int *__restrict__ bin_first,
             unsigned *__restrict__ amask, const int *__restrict__ words, const int *__restrict__ n_words,
             int *__restrict__ tslot, const int *__restrict__ run_slot0, const int *__restrict__ run_nent,
             const int *__restrict__ n_runs)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const int np = *n_prev, nw = *n_words, nr = *n_runs;
    if (bin_first) for (int i = tid; i < np; i += stride) bin_first[skey_prev[i]] = -1;
    for (int i = tid; i < nw; i += stride) amask[words[i]] = 0u;
    for (int r = tid; r < nr; r += stride) {
        const int s0 = run_slot0[r], ne = run_nent[r];
        for (int j = 0; j < ne; ++j) tslot[s0 + j] = -1;
    }
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
// A "run" is a maximal stretch of sorted markers in one lattice row (same cy, cz) whose owning
// cells are less than 4 apart in x, i.e. whose stencils chain together along x.  Runs of one row
// never touch the same cell, and a marker of source row (cy, cz) reaches the 16 target rows
// (cy-1+jy, cz-1+jz).  Stage A sweeps every run once, in sorted order, and produces for each of the
// 16 (jy, jz) offsets the x-profile  T[entry][jy*4+jz] = sum_k v_k w_y(jy) w_z(jz) w_x(X - cx_k + 1)
// over the run's x extent (entries cx_first-1 .. cx_last+2).  Stage B lets every active cell add
// up, in fixed order, the <= 16 profiles that reach it (one per source row).  All sums have a fixed
// order, so the result is bitwise reproducible.

struct RunTable {
    int *first, *end;   // sorted-marker range [first, end) of the run
    int *base;          // first T entry of the run
    int *slot0;         // index into tslot of the run's first entry
    int *nent;          // number of entries = cx_last - cx_first + 4
};

// tslot is a dense map [row][X + 1], X = -1 .. nx+1 (unwrapped x, so that runs at a periodic seam
// keep their own entries), holding the T entry or -1.
__device__ __forceinline__ int tslot_pitch(const Geom &g) { return g.nx + 3; }

// a3 (second part): one bit per sorted marker, set where a run starts.  Bits at and beyond n are
// set as well, so a forward search for the next run start always terminates.
__global__ void __launch_bounds__(256)
k_run_heads(const unsigned *__restrict__ skey, int n, Geom g, unsigned *__restrict__ headbits)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool head = true;
    if (i > 0 && i < n) {
        const unsigned key = skey[i], pk = skey[i - 1];
        const int row = (int)(key / (unsigned)g.nx), prow = (int)(pk / (unsigned)g.nx);
        head = (prow != row) || (((int)key - row * g.nx) - ((int)pk - prow * g.nx) >= 4);
    }
    const unsigned vote = __ballot_sync(0xffffffffu, head);
    if ((threadIdx.x & 31) == 0) headbits[i >> 5] = vote;
}

// set the bits x0..x1 (inclusive, 0 <= x0 <= x1 < nx) of one row of the active-cell mask; the
// thread that turns a word non-zero appends it to the word list
__device__ __forceinline__ void mark_span(unsigned *__restrict__ amask, int rowbase, int x0, int x1,
                                          int *__restrict__ words, int *__restrict__ n_words)
{
    for (int w = x0 >> 5; w <= (x1 >> 5); ++w) {
        const int lo = max(x0 - (w << 5), 0), hi = min(x1 - (w << 5), 31);
        const unsigned bits = (0xffffffffu >> (31 - hi)) & (0xffffffffu << lo);
        if (atomicOr(amask + rowbase + w, bits) == 0u) {
            const unsigned act = __activemask();
            const int lane = threadIdx.x & 31;
            const int leader = __ffs(act) - 1;
            int base = 0;
            if (lane == leader) base = atomicAdd(n_words, __popc(act));
            base = __shfl_sync(act, base, leader);
            words[base + __popc(act & ((1u << lane) - 1u))] = rowbase + w;
        }
    }
}

// a3 (third part): the first marker of every run finds the run's end and takes a block of T entries.
__global__ void __launch_bounds__(256)
k_runs(const unsigned *__restrict__ skey, int n, Geom g, const unsigned *__restrict__ headbits, RunTable rt,
       int *__restrict__ n_runs, int *__restrict__ t_count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const unsigned myword = (i < n) ? headbits[i >> 5] : 0u;
    const bool head = (myword >> lane) & 1u;
    int row = 0, cx = 0, end = 0, nent = 0;
    if (head) {
        // next set bit after i
        int wi = i >> 5;
        unsigned w = (lane == 31) ? 0u : (myword & (0xffffffffu << (lane + 1)));
        while (w == 0u) w = headbits[++wi];
        end = (wi << 5) + __ffs(w) - 1;
        if (end > n) end = n;
        const unsigned key = skey[i], lk = skey[end - 1];
        row = (int)(key / (unsigned)g.nx);
        cx = (int)key - row * g.nx;
        nent = ((int)lk - row * g.nx) - cx + 4;
    }
    const unsigned vote = __ballot_sync(0xffffffffu, head);
    if (!vote) return;
    int incl = nent;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    int rbase = 0, tbase = 0;
    if (lane == 0) { rbase = atomicAdd(n_runs, __popc(vote)); tbase = atomicAdd(t_count, total); }
    rbase = __shfl_sync(0xffffffffu, rbase, 0);
    tbase = __shfl_sync(0xffffffffu, tbase, 0);
    if (!head) return;
    const int r = rbase + __popc(vote & ((1u << lane) - 1u));
    const int base = tbase + incl - nent;
    const int s0 = row * tslot_pitch(g) + cx;        // X = cx - 1  ->  column X + 1 = cx
    rt.first[r] = i; rt.end[r] = end; rt.base[r] = base; rt.slot0[r] = s0; rt.nent[r] = nent;
}

// a3 (fourth part): one half-warp per run publishes the run: its T entries go into tslot and its
// cells -- the whole x span cx_first-1 .. cx_last+2 in each of the 16 target rows, one row per lane
// -- are marked in the active-cell bitmask.
__global__ void __launch_bounds__(256)
k_run_publish(Geom g, RunTable rt, const int *__restrict__ n_runs, int *__restrict__ tslot,
              unsigned *__restrict__ amask, int *__restrict__ words, int *__restrict__ n_words)
{
    const int l = threadIdx.x & 15;
    const int hw = (blockIdx.x * blockDim.x + threadIdx.x) >> 4;
    const int nhw = (gridDim.x * blockDim.x) >> 4;
    const int nr = *n_runs;
    const int pitch = tslot_pitch(g);
    for (int r = hw; r < nr; r += nhw) {
        const int s0 = rt.slot0[r], nent = rt.nent[r], base = rt.base[r];
        for (int j = l; j < nent; j += 16) tslot[s0 + j] = base + j;
        const int row = s0 / pitch;
        const int cx = s0 - row * pitch;
        const int cz = row / g.ny, cy = row - cz * g.ny;
        // x span [cx-1, cx+nent-2], wrapped on a periodic axis (inside the box on a wall axis)
        const int xa = cx - 1, xb = cx + nent - 2;
        int x0a, x1a, x0b = 0, x1b = -1;
        if (nent >= g.nx) { x0a = 0; x1a = g.nx - 1; }
        else if (xa < 0) { x0a = xa + g.nx; x1a = g.nx - 1; x0b = 0; x1b = xb; }
        else if (xb >= g.nx) { x0a = xa; x1a = g.nx - 1; x0b = 0; x1b = xb - g.nx; }
        else { x0a = xa; x1a = xb; }
        const int y = wrap(cy - 1 + (l >> 2), g.ny);
        const int z = wrap(cz - 1 + (l & 3), g.nz);
        const int rowbase = (z * g.ny + y) * g.nxw;
        mark_span(amask, rowbase, x0a, x1a, words, n_words);
        if (x1b >= x0b) mark_span(amask, rowbase, x0b, x1b, words, n_words);
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

// Stage A: one half-warp per run, lane l = jy*4 + jz owns the profile of target-row offset (jy, jz)
// and keeps a sliding window of four x cells (cxw-1 .. cxw+2) in registers; cells that fall out of
// the window as the sweep advances are final and are written to T (16 lanes x float4 = 256 B).
// Runs are handed out through an atomic cursor (they differ a lot in length); the data of marker
// i+1 is fetched while marker i is accumulated.
struct Acc3 { float x, y, z; };

__global__ void __launch_bounds__(256)
k_spread_rows(RunTable rt, const int *__restrict__ n_runs, int *__restrict__ cursor,
              const float4 *__restrict__ wx4, const float *__restrict__ wyz16, const float4 *__restrict__ val,
              float4 *__restrict__ T)
{
    const int lane = threadIdx.x & 31;
    const int l = lane & 15;
    const unsigned hmask = 0xffffu << (lane & 16);
    const int nr = *n_runs;
    for (;;) {
        int r = 0;
        if (l == 0) r = atomicAdd(cursor, 1);
        r = __shfl_sync(hmask, r, lane & 16);
        if (r >= nr) break;
        const int i0 = rt.first[r], i1 = rt.end[r];
        float4 *out = T + (size_t)rt.base[r] * 16 + l;
        Acc3 a0{0.f, 0.f, 0.f}, a1{0.f, 0.f, 0.f}, a2{0.f, 0.f, 0.f}, a3{0.f, 0.f, 0.f};
        // markers are taken in batches of RB: all loads of a batch are issued before the first
        // marker is accumulated, so the memory latency is paid once per batch, not once per marker
        constexpr int RB = 4;
        int cxw = __float_as_int(val[i0].w);
        for (int ib = i0; ib < i1; ib += RB) {
            float4 bv[RB], bw[RB];
            float bz[RB];
#pragma unroll
            for (int j = 0; j < RB; ++j) {
                const int i = min(ib + j, i1 - 1);
                bv[j] = val[i];
                bw[j] = wx4[i];
                bz[j] = wyz16[(size_t)i * 16 + l];
            }
#pragma unroll
            for (int j = 0; j < RB; ++j) {
                if (ib + j < i1) {
                    const float4 v = bv[j], w = bw[j];
                    const int cx = __float_as_int(v.w);
                    if (cx != cxw) {
                        // the window moves right by 1..3 cells: its leftmost cells are complete
                        const int sh = cx - cxw;
                        out[0] = make_float4(a0.x, a0.y, a0.z, 0.f);
                        if (sh > 1) out[16] = make_float4(a1.x, a1.y, a1.z, 0.f);
                        if (sh > 2) out[32] = make_float4(a2.x, a2.y, a2.z, 0.f);
                        const Acc3 zero{0.f, 0.f, 0.f};
                        const Acc3 b0 = sh == 1 ? a1 : (sh == 2 ? a2 : a3);
                        const Acc3 b1 = sh == 1 ? a2 : (sh == 2 ? a3 : zero);
                        const Acc3 b2 = sh == 1 ? a3 : zero;
                        a0 = b0; a1 = b1; a2 = b2; a3 = zero;
                        out += 16 * sh;
                        cxw = cx;
                    }
                    const float vx = v.x * bz[j], vy = v.y * bz[j], vz = v.z * bz[j];
                    a0.x = fmaf(w.x, vx, a0.x); a0.y = fmaf(w.x, vy, a0.y); a0.z = fmaf(w.x, vz, a0.z);
                    a1.x = fmaf(w.y, vx, a1.x); a1.y = fmaf(w.y, vy, a1.y); a1.z = fmaf(w.y, vz, a1.z);
                    a2.x = fmaf(w.z, vx, a2.x); a2.y = fmaf(w.z, vy, a2.y); a2.z = fmaf(w.z, vz, a2.z);
                    a3.x = fmaf(w.w, vx, a3.x); a3.y = fmaf(w.w, vy, a3.y); a3.z = fmaf(w.w, vz, a3.z);
                }
            }
        }
        out[0] = make_float4(a0.x, a0.y, a0.z, 0.f);
        out[16] = make_float4(a1.x, a1.y, a1.z, 0.f);
        out[32] = make_float4(a2.x, a2.y, a2.z, 0.f);
        out[48] = make_float4(a3.x, a3.y, a3.z, 0.f);
    }
}

// Stage B: one thread per active cell: add the profiles of the source rows (y+1-jy, z+1-jz) at this
// x, jy and jz ascending (fixed order).
//   LAST = false:  U^{m+1}(X) = U^m(X) + sum   (R8)      LAST = true:  G(X) = sum
template <bool LAST>
__global__ void __launch_bounds__(256)
k_spread_collect(Geom g, const int *__restrict__ tslot, const float4 *__restrict__ T,
                 const int *__restrict__ cells, const int *__restrict__ n_cells, float4 *__restrict__ field)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const int nc = *n_cells;
    const int pitch = tslot_pitch(g);
    for (int k = tid; k < nc; k += stride) {
        const int cell = __ldg(cells + k);
        const int row = cell / g.nx;
        const int x = cell - row * g.nx;
        const int z = row / g.ny, y = row - z * g.ny;
        // ghost columns of a periodic x axis: X = x + nx (for x <= 1) and X = -1 (for x = nx-1)
        const int ghost = g.wallx ? -1 : (x <= 1 ? x + g.nx + 1 : (x == g.nx - 1 ? 0 : -1));
        float sx = 0.f, sy = 0.f, sz = 0.f;
#pragma unroll
        for (int jy = 0; jy < 4; ++jy) {
            int cy = y + 1 - jy;
            if (g.wally) { if (cy < 0 || cy >= g.ny) continue; } else cy = wrap(cy, g.ny);
#pragma unroll
            for (int jz = 0; jz < 4; ++jz) {
                int cz = z + 1 - jz;
                if (g.wallz) { if (cz < 0 || cz >= g.nz) continue; } else cz = wrap(cz, g.nz);
                const int *trow = tslot + (size_t)(cz * g.ny + cy) * pitch;
                const int e = __ldg(trow + x + 1);
                if (e >= 0) {
                    const float4 t = T[(size_t)e * 16 + (jy * 4 + jz)];
                    sx += t.x; sy += t.y; sz += t.z;
                }
                if (ghost >= 0) {
                    const int e2 = __ldg(trow + ghost);
                    if (e2 >= 0) {
                        const float4 t = T[(size_t)e2 * 16 + (jy * 4 + jz)];
                        sx += t.x; sy += t.y; sz += t.z;
                    }
                }
            }
        }
        if (LAST) {
            field[cell] = make_float4(sx, sy, sz, 0.f);
        } else {
            float4 u = field[cell];
            u.x += sx; u.y += sy; u.z += sz;
            field[cell] = u;
        }
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

}  // namespace lbmk
