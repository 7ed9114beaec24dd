// Lattice kernels: fused pull-stream + BGK collide + force (row a8 of SURVEY.md section 8),
// moments on active cells (a4), field initialisation and canonical read-out (a9).
//
// Storage: two SoA buffers of 19 fp32 planes, plane i = df_i[z][y][x] (x fastest).  A buffer
// holds POST-collision populations (R19); the canonical (post-stream, pre-collision) state of
// P:31 is what a pull from that buffer yields:
//     f_i(x, n+1) = f'_i(x - e_i)                       eq. (4), P:49 (indices wrapped if periodic)
//     f_i(x, n+1) = f'_{opp i}(x)   if x - e_i lies behind a wall face (half-way bounce-back, R16)
#pragma once
#include "d3q19.cuh"

// cache operators of the population streams (each value is read once and written once per step);
// the modes exist for measurement builds, the defaults are the ones measured fastest.
#ifndef LBM_LD_MODE
#define LBM_LD_MODE 0
#endif
#ifndef LBM_ST_MODE
#define LBM_ST_MODE 1
#endif
#if LBM_LD_MODE == 1
#define LBM_LOAD(p) __ldcs(p)
#elif LBM_LD_MODE == 2
#define LBM_LOAD(p) __ldlu(p)
#elif LBM_LD_MODE == 3
#define LBM_LOAD(p) __ldcg(p)
#elif LBM_LD_MODE == 4
#define LBM_LOAD(p) (*(p))
#else
#define LBM_LOAD(p) __ldg(p)
#endif
#if LBM_ST_MODE == 1
#define LBM_STORE(p, v) (*(p) = (v))      /* plain write-back stores: measured 2-3 % faster than .cs */
#elif LBM_ST_MODE == 2
#define LBM_STORE(p, v) __stcg(p, v)
#elif LBM_ST_MODE == 3
#define LBM_STORE(p, v) __stwt(p, v)
#else
#define LBM_STORE(p, v) __stcs(p, v)
#endif

namespace lbmk {

// CS = cache-streaming (evict-first) accesses: for the bulk pass that runs BESIDE the MDF loop, so that the ~1 GB it
// streams through L2 does not evict the few MB the MDF kernels work on (U, the footprints, the markers)
template <bool CS> __device__ __forceinline__ float lbm_load(const float *p) { return CS ? __ldcs(p) : LBM_LOAD(p); }
template <bool CS> __device__ __forceinline__ void lbm_store(float *p, float v) { if (CS) __stcs(p, v); else LBM_STORE(p, v); }

struct Geom {
    int nx, ny, nz;
    int nxw;             // 32-cell words per x-row of the active-cell bitmask
    long long cells;
    long long pitch;     // floats between two population planes (>= cells; padding staggers the
                         // 19 read and 19 write streams over the memory channels)
    int wallx, wally, wallz;
};

// The neighbourhood of one cell for the pull: wrapped neighbour coordinates and, per axis, whether
// stepping -1 / +1 leaves the domain through a wall.
struct Nbr {
    int xm, xp, ym, yp, zm, zp;
    bool wxm, wxp, wym, wyp, wzm, wzp;
};

__device__ __forceinline__ Nbr neighbours(const Geom &g, int x, int y, int z)
{
    Nbr n;
    n.xm = (x == 0) ? g.nx - 1 : x - 1;
    n.xp = (x == g.nx - 1) ? 0 : x + 1;
    n.ym = (y == 0) ? g.ny - 1 : y - 1;
    n.yp = (y == g.ny - 1) ? 0 : y + 1;
    n.zm = (z == 0) ? g.nz - 1 : z - 1;
    n.zp = (z == g.nz - 1) ? 0 : z + 1;
    n.wxm = g.wallx && x == 0;
    n.wxp = g.wallx && x == g.nx - 1;
    n.wym = g.wally && y == 0;
    n.wyp = g.wally && y == g.ny - 1;
    n.wzm = g.wallz && z == 0;
    n.wzp = g.wallz && z == g.nz - 1;
    return n;
}

// Pull the 19 canonical populations of cell (x,y,z) out of a post-collision buffer.
template <bool CS = false>
__device__ __forceinline__ void pull_cell(const float *__restrict__ src, const Geom &g, const Nbr &n, int x, int y,
                                          int z, float (&df)[NQ])
{
    const size_t cells = (size_t)g.pitch;
    const int self = (z * g.ny + y) * g.nx + x;
#pragma unroll
    for (int i = 0; i < NQ; ++i) {
        // source cell x - e_i
        const int sx = dir_ex(i) == 1 ? n.xm : (dir_ex(i) == -1 ? n.xp : x);
        const int sy = dir_ey(i) == 1 ? n.ym : (dir_ey(i) == -1 ? n.yp : y);
        const int sz = dir_ez(i) == 1 ? n.zm : (dir_ez(i) == -1 ? n.zp : z);
        bool behind_wall = false;
        if (dir_ex(i) == 1) behind_wall |= n.wxm;
        if (dir_ex(i) == -1) behind_wall |= n.wxp;
        if (dir_ey(i) == 1) behind_wall |= n.wym;
        if (dir_ey(i) == -1) behind_wall |= n.wyp;
        if (dir_ez(i) == 1) behind_wall |= n.wzm;
        if (dir_ez(i) == -1) behind_wall |= n.wzp;
        const int cell = behind_wall ? self : (sz * g.ny + sy) * g.nx + sx;
        const int plane = behind_wall ? dir_opp(i) : i;
        df[i] = lbm_load<CS>(src + (size_t)plane * cells + cell);
    }
}

__device__ __forceinline__ bool cell_is_active(const unsigned *__restrict__ amask, const Geom &g, int x, int y, int z)
{
    const unsigned w = __ldg(amask + (size_t)(z * g.ny + y) * g.nxw + (x >> 5));
    return (w >> (x & 31)) & 1u;
}

// Byte offsets of the interior pull and of the stores, the same for every interior cell; filled on
// the host (plane_offsets) so that each access costs one 64-bit add of a constant-bank operand.
struct PlaneOffsets {
    long long ld[NQ];    // (i pitch - e_y nx - e_z nx ny) * 4: source of direction i relative to the cell (x handled apart)
    long long st[NQ];    // (i pitch) * 4
};

inline PlaneOffsets plane_offsets(const Geom &g)
{
    PlaneOffsets o;
    for (int i = 0; i < NQ; ++i) {
        o.ld[i] = 4 * ((long long)i * g.pitch - (long long)dir_ey(i) * g.nx - (long long)dir_ez(i) * g.nx * g.ny);
        o.st[i] = 4 * ((long long)i * g.pitch);
    }
    return o;
}

// Pull for a cell whose y and z neighbours are plain lattice rows (no wrap, no wall) and that has
// no x wall behind it: every source sits at a kernel-uniform byte offset (plane + row shift) from
// one of three per-thread pointers (the cell itself, its wrapped x-1 and x+1 neighbours).
template <bool CS = false>
__device__ __forceinline__ void pull_cell_inner(const float *__restrict__ src, const Geom &g, const PlaneOffsets &po,
                                                int x, int self, float (&df)[NQ])
{
    const char *__restrict__ p0 = reinterpret_cast<const char *>(src + self);
    const char *__restrict__ pm = p0 + 4 * ((x == 0) ? g.nx - 1 : -1);          // cell at x-1 (wrapped)
    const char *__restrict__ pp = p0 + 4 * ((x == g.nx - 1) ? 1 - g.nx : 1);    // cell at x+1 (wrapped)
#pragma unroll
    for (int i = 0; i < NQ; ++i) {
        const char *__restrict__ b = dir_ex(i) == 1 ? pm : (dir_ex(i) == -1 ? pp : p0);
        df[i] = lbm_load<CS>(reinterpret_cast<const float *>(b + po.ld[i]));
    }
}

// ---------------------------------------------------------------------------------------------
// a8, one thread per cell, x along threadIdx.x (coalesced 128 B per warp and plane), one x-row
// segment per block so that "is this an interior row" is block-uniform.
//   MODE 0: pure LBM (a = g_body everywhere).
//   MODE 1: fused IBM pass: one bitmask word per warp, G read only where a marker stencil reaches
//           (both issued before the population loads so their latency overlaps).
//   MODE 2: bulk pass of the overlapped step: a warp covers exactly the 32 cells of one mask word;
//           warps whose word is non-zero are SKIPPED as a whole (k_stream_collide_words updates
//           them once G is known), so both passes write whole 128-byte lines (measured: skipping
//           8-cell groups instead leaves less for the second pass but is slower overall).
//           Everywhere else a = g_body: this pass needs nothing from the IBM and runs beside it.
enum { LBM_PURE = 0, LBM_FUSED = 1, LBM_BULK = 2 };

template <int MODE, int THREADS, int MINB, bool CS = false>
__global__ void __launch_bounds__(THREADS, MINB)
k_stream_collide_scalar(const float *__restrict__ src, float *__restrict__ dst, const __grid_constant__ Geom g,
                        const __grid_constant__ CollisionConst cc, const __grid_constant__ PlaneOffsets po,
                        const unsigned *__restrict__ amask, const float4 *__restrict__ G)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.nx || y >= g.ny) return;
    const int self = (z * g.ny + y) * g.nx + x;

    float ax = cc.gbx, ay = cc.gby, az = cc.gbz;
    if (MODE == LBM_FUSED) {
        if (cell_is_active(amask, g, x, y, z)) {
            const float4 gv = __ldg(G + self);
            ax += gv.x; ay += gv.y; az += gv.z;
        }
    }
    if (MODE == LBM_BULK) {
        if (__ldg(amask + (size_t)(z * g.ny + y) * g.nxw + (x >> 5)) != 0u) return;
    }
    float df[NQ];
    const bool xwall = g.wallx && (x == 0 || x == g.nx - 1);
    if (y > 0 && y < g.ny - 1 && z > 0 && z < g.nz - 1 && !xwall) {
        pull_cell_inner<CS>(src, g, po, x, self, df);
    } else {
        const Nbr n = neighbours(g, x, y, z);
        pull_cell<CS>(src, g, n, x, y, z, df);
    }
    collide(df, ax, ay, az, cc);
    char *__restrict__ q = reinterpret_cast<char *>(dst + self);
#pragma unroll
    for (int i = 0; i < NQ; ++i) lbm_store<CS>(reinterpret_cast<float *>(q + po.st[i]), df[i]);
}

// a8 on the words the bulk pass skipped (second pass of the overlapped step): one warp per entry of
// the active-word list, lane = cell of the word; a = G + g_body where the cell's bit is set, g_body
// on the other cells of the word.
// the words pass of one warp team: warp `warp` of `nwarps` takes the entries warp, warp + nwarps, ... of the list
__device__ __forceinline__ void stream_collide_words(const float *__restrict__ src, float *__restrict__ dst, const Geom &g,
                                                     const CollisionConst &cc, const PlaneOffsets &po,
                                                     const unsigned *__restrict__ amask, const int *__restrict__ words,
                                                     const int nw, const float4 *__restrict__ G, const int warp,
                                                     const int nwarps, const int lane)
{
    // the word and its mask bits of the next round are fetched while this round's cells are updated
    int w_next = warp < nw ? __ldg(words + warp) : 0;
    unsigned bits_next = warp < nw ? __ldg(amask + w_next) : 0u;
    for (int k = warp; k < nw; k += nwarps) {
        const int w = w_next;
        const unsigned bits = bits_next;
        if (k + nwarps < nw) {
            w_next = __ldg(words + k + nwarps);
            bits_next = __ldg(amask + w_next);
        }
        const int row = w / g.nxw;
        const int x = (w - row * g.nxw) * 32 + lane;
        if (x >= g.nx) continue;
        const int z = row / g.ny, y = row - z * g.ny;
        const int self = row * g.nx + x;
        float ax = cc.gbx, ay = cc.gby, az = cc.gbz;
        if ((bits >> lane) & 1u) {
            const float4 gv = __ldcg(G + self);          // written earlier in the step, possibly by this very kernel
            ax += gv.x; ay += gv.y; az += gv.z;
        }
        float df[NQ];
        const bool xwall = g.wallx && (x == 0 || x == g.nx - 1);
        if (y > 0 && y < g.ny - 1 && z > 0 && z < g.nz - 1 && !xwall) {
            pull_cell_inner(src, g, po, x, self, df);
        } else {
            const Nbr n = neighbours(g, x, y, z);
            pull_cell(src, g, n, x, y, z, df);
        }
        collide(df, ax, ay, az, cc);
        char *__restrict__ q = reinterpret_cast<char *>(dst + self);
#pragma unroll
        for (int i = 0; i < NQ; ++i) LBM_STORE(reinterpret_cast<float *>(q + po.st[i]), df[i]);
    }
}

__global__ void __launch_bounds__(256)
k_stream_collide_words(const float *__restrict__ src, float *__restrict__ dst, const __grid_constant__ Geom g,
                       const __grid_constant__ CollisionConst cc, const __grid_constant__ PlaneOffsets po,
                       const unsigned *__restrict__ amask, const int *__restrict__ words,
                       const int *__restrict__ n_words, const float4 *__restrict__ G, long long *__restrict__ step_ctr)
{
    // last kernel of a coupled step: advance the device-side time-step counter (read by k_kinematics)
    if (step_ctr && blockIdx.x == 0 && threadIdx.x == 0) *step_ctr += 1;
    stream_collide_words(src, dst, g, cc, po, amask, words, *n_words, G, (blockIdx.x * blockDim.x + threadIdx.x) >> 5,
                         (gridDim.x * blockDim.x) >> 5, threadIdx.x & 31);
}

// ---------------------------------------------------------------------------------------------
// a8, vectorised variant: one thread per 4 consecutive x cells; every plane is read and written
// with 128-bit accesses.  Directions with e_x = 0 are plain aligned float4 loads of the source
// row; directions with e_x = +-1 need the row shifted by one cell: three of the four values come
// from the thread's own aligned float4 and the fourth from the neighbouring lane's float4 via a
// warp shuffle (lanes at a warp or row edge fetch that one value with a scalar load instead).
// Requires nx % 4 == 0.
template <bool IBM>
__global__ void __launch_bounds__(256)
k_stream_collide_vec4(const float *__restrict__ src, float *__restrict__ dst, Geom g, CollisionConst cc,
                      const unsigned *__restrict__ amask, const float4 *__restrict__ G)
{
    const int nx4 = g.nx >> 2;
    const int x4 = blockIdx.x * blockDim.x + threadIdx.x;   // index of the 4-cell group in the row
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    const bool live = (x4 < nx4) && (y < g.ny);
    const size_t cells = (size_t)g.pitch;
    const unsigned lane = (threadIdx.y * blockDim.x + threadIdx.x) & 31u;

    // clamp dead threads onto a valid cell so that shuffles stay convergent; they do not store
    const int xg = live ? x4 : 0;
    const int yy = live ? y : 0;
    const int x0 = xg << 2;
    const Nbr n = neighbours(g, x0, yy, z);   // y/z neighbours and wall flags of the row
    const bool wall_lo = g.wallx && x0 == 0;             // cell x0 has the low-x wall behind it
    const bool wall_hi = g.wallx && x0 + 4 == g.nx;      // cell x0+3 has the high-x wall behind it
    const int self = (z * g.ny + yy) * g.nx + x0;

    // do my lane neighbours hold the adjacent 4-cell groups of the same row?
    const int lane_x4_dn = __shfl_up_sync(0xffffffffu, xg, 1);
    const int lane_y_dn = __shfl_up_sync(0xffffffffu, yy, 1);
    const int lane_x4_up = __shfl_down_sync(0xffffffffu, xg, 1);
    const int lane_y_up = __shfl_down_sync(0xffffffffu, yy, 1);
    const bool have_dn = lane > 0 && lane_x4_dn == xg - 1 && lane_y_dn == yy;
    const bool have_up = lane < 31 && lane_x4_up == xg + 1 && lane_y_up == yy;

    float df[4][NQ];
#pragma unroll
    for (int i = 0; i < NQ; ++i) {
        const int sy = dir_ey(i) == 1 ? n.ym : (dir_ey(i) == -1 ? n.yp : yy);
        const int sz = dir_ez(i) == 1 ? n.zm : (dir_ez(i) == -1 ? n.zp : z);
        bool row_behind_wall = false;       // the whole source row lies behind a y or z wall
        if (dir_ey(i) == 1) row_behind_wall |= n.wym;
        if (dir_ey(i) == -1) row_behind_wall |= n.wyp;
        if (dir_ez(i) == 1) row_behind_wall |= n.wzm;
        if (dir_ez(i) == -1) row_behind_wall |= n.wzp;
        if (dir_ex(i) == 0) {
            const int cell = row_behind_wall ? self : (sz * g.ny + sy) * g.nx + x0;
            const int plane = row_behind_wall ? dir_opp(i) : i;
            const float4 v = __ldg(reinterpret_cast<const float4 *>(src + (size_t)plane * cells + cell));
            df[0][i] = v.x; df[1][i] = v.y; df[2][i] = v.z; df[3][i] = v.w;
        } else {
            // bounce-back rows read plane opp(i) at the cell itself (no x shift); regular rows
            // read plane i shifted by -e_x.
            const int rowbase = row_behind_wall ? (z * g.ny + yy) * g.nx : (sz * g.ny + sy) * g.nx;
            const int plane = row_behind_wall ? dir_opp(i) : i;
            const float *__restrict__ p = src + (size_t)plane * cells + rowbase;
            const float4 v = __ldg(reinterpret_cast<const float4 *>(p + x0));
            if (dir_ex(i) == 1) {
                // regular: cells x0..x0+3 take p[x0-1 .. x0+2]
                float edge = __shfl_up_sync(0xffffffffu, v.w, 1);
                if (!have_dn) edge = __ldg(p + n.xm);
                float a0 = edge, a1 = v.x, a2 = v.y, a3 = v.z;
                if (row_behind_wall) { a0 = v.x; a1 = v.y; a2 = v.z; a3 = v.w; }
                else if (wall_lo) a0 = __ldg(src + (size_t)dir_opp(i) * cells + self);
                df[0][i] = a0; df[1][i] = a1; df[2][i] = a2; df[3][i] = a3;
            } else {
                // regular: cells x0..x0+3 take p[x0+1 .. x0+4]
                float edge = __shfl_down_sync(0xffffffffu, v.x, 1);
                const int xp3 = (x0 + 4 == g.nx) ? 0 : x0 + 4;
                if (!have_up) edge = __ldg(p + xp3);
                float a0 = v.y, a1 = v.z, a2 = v.w, a3 = edge;
                if (row_behind_wall) { a0 = v.x; a1 = v.y; a2 = v.z; a3 = v.w; }
                else if (wall_hi) a3 = __ldg(src + (size_t)dir_opp(i) * cells + self + 3);
                df[0][i] = a0; df[1][i] = a1; df[2][i] = a2; df[3][i] = a3;
            }
        }
    }
    if (!live) return;

    float ax[4], ay[4], az[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) { ax[c] = cc.gbx; ay[c] = cc.gby; az[c] = cc.gbz; }
    if (IBM) {
        const unsigned w = __ldg(amask + (size_t)(z * g.ny + yy) * g.nxw + (x0 >> 5));
        const unsigned bits = (w >> (x0 & 31)) & 0xFu;
        if (bits) {
#pragma unroll
            for (int c = 0; c < 4; ++c)
                if ((bits >> c) & 1u) {
                    const float4 gv = __ldg(G + self + c);
                    ax[c] += gv.x; ay[c] += gv.y; az[c] += gv.z;
                }
        }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) collide(df[c], ax[c], ay[c], az[c], cc);
#pragma unroll
    for (int i = 0; i < NQ; ++i)
        __stcs(reinterpret_cast<float4 *>(dst + (size_t)i * cells + self),
               make_float4(df[0][i], df[1][i], df[2][i], df[3][i]));
}

// ---------------------------------------------------------------------------------------------
// R18: f = Eq(rho0, u0) as the canonical state, stored so that the pull of the next step (and of
// the read-out) recovers it: the value f_i(x) goes to plane i of cell x - e_i, or, when that cell
// lies behind a wall, to plane opp(i) of x itself (the inverse of the two pull rules above).
__global__ void __launch_bounds__(256)
k_init_fields(float *__restrict__ buf, Geom g, const float *__restrict__ rho0, const float *__restrict__ u0)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.nx || y >= g.ny) return;
    const size_t cells = (size_t)g.cells;
    const size_t pitch = (size_t)g.pitch;
    const int self = (z * g.ny + y) * g.nx + x;
    const float drho = rho0 ? (rho0[self] - 1.0f) : 0.0f;
    const float ux = u0 ? u0[self] : 0.0f;
    const float uy = u0 ? u0[cells + self] : 0.0f;
    const float uz = u0 ? u0[2 * cells + self] : 0.0f;
    const Nbr n = neighbours(g, x, y, z);
#pragma unroll
    for (int i = 0; i < NQ; ++i) {
        const int sx = dir_ex(i) == 1 ? n.xm : (dir_ex(i) == -1 ? n.xp : x);
        const int sy = dir_ey(i) == 1 ? n.ym : (dir_ey(i) == -1 ? n.yp : y);
        const int sz = dir_ez(i) == 1 ? n.zm : (dir_ez(i) == -1 ? n.zp : z);
        bool behind_wall = false;
        if (dir_ex(i) == 1) behind_wall |= n.wxm;
        if (dir_ex(i) == -1) behind_wall |= n.wxp;
        if (dir_ey(i) == 1) behind_wall |= n.wym;
        if (dir_ey(i) == -1) behind_wall |= n.wyp;
        if (dir_ez(i) == 1) behind_wall |= n.wzm;
        if (dir_ez(i) == -1) behind_wall |= n.wzp;
        const int cell = behind_wall ? self : (sz * g.ny + sy) * g.nx + sx;
        const int plane = behind_wall ? dir_opp(i) : i;
        buf[(size_t)plane * pitch + cell] = equilibrium_dev(i, drho, ux, uy, uz);
    }
}

// a9 / O8: canonical rho, bare U (eq. (1)) of every cell; force = G where a stencil reached in
// the last step, zero elsewhere.  Output planes [nz][ny][nx]; any output may be NULL.
__global__ void __launch_bounds__(256)
k_read_fields(const float *__restrict__ src, Geom g, const unsigned *__restrict__ amask_last,
              const float4 *__restrict__ G, float *__restrict__ rho, float *__restrict__ u, float *__restrict__ force)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= g.nx || y >= g.ny) return;
    const size_t cells = (size_t)g.cells;
    const int self = (z * g.ny + y) * g.nx + x;
    if (rho || u) {
        const Nbr n = neighbours(g, x, y, z);
        float df[NQ], drho, ux, uy, uz;
        pull_cell(src, g, n, x, y, z, df);
        moments(df, drho, ux, uy, uz);
        if (rho) rho[self] = 1.0f + drho;
        if (u) { u[self] = ux; u[cells + self] = uy; u[2 * cells + self] = uz; }
    }
    if (force) {
        float4 gv = make_float4(0.f, 0.f, 0.f, 0.f);
        if (amask_last && cell_is_active(amask_last, g, x, y, z)) gv = G[self];
        force[self] = gv.x; force[cells + self] = gv.y; force[2 * cells + self] = gv.z;
    }
}

// a4: rho, U of eq. (1) for the active cells only (the paper's "kernel strategy", P:215,
// de-duplicated): one thread per entry of the active-cell list pulls its 19 populations.
// U is stored as float4 (Ux, Uy, Uz, rho).
__global__ void __launch_bounds__(256)
k_moments_active(const float *__restrict__ src, const __grid_constant__ Geom g,
                 const __grid_constant__ PlaneOffsets po, const int *__restrict__ cells,
                 const int *__restrict__ n_cells, float4 *__restrict__ U)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const int nc = *n_cells;
    for (int k = tid; k < nc; k += stride) {
        const int cell = __ldg(cells + k);
        const int row = cell / g.nx;
        const int x = cell - row * g.nx;
        const int z = row / g.ny, y = row - z * g.ny;
        float df[NQ], drho, ux, uy, uz;
        const bool xwall = g.wallx && (x == 0 || x == g.nx - 1);
        if (y > 0 && y < g.ny - 1 && z > 0 && z < g.nz - 1 && !xwall) {
            pull_cell_inner(src, g, po, x, cell, df);
        } else {
            const Nbr n = neighbours(g, x, y, z);
            pull_cell(src, g, n, x, y, z, df);
        }
        moments(df, drho, ux, uy, uz);
        U[cell] = make_float4(ux, uy, uz, 1.0f + drho);
    }
}

}  // namespace lbmk
