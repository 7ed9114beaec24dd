// The multi-direct-forcing loop as the product path runs it: per iteration ONE tile pass
// that interpolates (a5), corrects (a6) and spreads (a7, stage A) and one collect pass (a7, stage B).
//
//   tile pass   one warp per tile (the chunks of one 8-cell x block whose source rows lie in one aligned
//               TR x TR block of (y, z), see ibm_kernels.cuh).  The warp stages the tile's window of U^m
//               -- (TR+3)^2 rows x (8+3) cells, every cell some marker of the tile can reach -- in ITS OWN
//               shared memory, then takes the tile's markers 32 at a time:
//                 phase 1, lane = marker: Peskin weights from the fractional position (3 square roots),
//                   u^m(k) from the window (64 shared-memory reads instead of 64 global gathers),
//                   g = u_k - u^m(k), Delta u += s g, and the marker's sweep record (value, x weights,
//                   16 y-z weights) goes to the warp's staging buffer;
//                 phase 2, lane = (half of the 4-cell x window, target-row offset (jy, jz)): the warp
//                   sweeps the 32 staged markers in sorted order; the window slides along x, finished
//                   cells are added to the tile's footprint in shared memory.
//               Every sum has a fixed order: no atomics, no block-level barrier, bitwise reproducible.
//               The value s g (or Delta u in the last iteration) never leaves the SM: the interpolation
//               kernel, its `sg` round trip and the per-marker weight tables of the round-1 pipeline
//               (96 B per marker and iteration) are gone; a marker costs 48 B read + 16 B written.
//   collect     one thread per active cell adds the footprint elements that hold the cell (fixed order).
//
// Small marker sets (a single propeller) run the whole loop -- moments, N x (tile pass, collect) -- as
// ONE persistent kernel with grid-wide barriers instead of 2N + 1 dependent launches, on tiles of a
// single source row (TR = 1) so that a few thousand markers still spread over all SMs.  That kernel also
// updates the lattice cells inside the stencils once G is complete, and it releases the lattice-wide
// stream-collide pass that runs beside it (its programmatic dependent) as soon as all its blocks are resident.
#pragma once
#include "ibm_kernels.cuh"

namespace lbmk {

#ifndef MDF_MIN_BLOCKS_CFG
#define MDF_MIN_BLOCKS_CFG 4
#endif
constexpr int MDF_WARPS = 4;            // warps per block of the tile pass
constexpr int MDF_MIN_BLOCKS = MDF_MIN_BLOCKS_CFG;   // register cap of the tile pass: 65536 / (128 threads x MDF_MIN_BLOCKS)
constexpr int MDF_BATCH = 32;           // markers per phase-1 / phase-2 round (= lanes)
constexpr int MDF_STAGE_RECS = MDF_BATCH + 1;        // one padding record: the sweep reads one record ahead
constexpr int MDF_STAGE_BYTES = (MDF_STAGE_RECS * 96 + 127) / 128 * 128;

struct MdfArgs {
    Geom g;
    ChunkGeom cg;
    TileGeom tg;
    // tiles of the marker set
    const int2 *tile_rec;        // [tile][TR*TR] sorted-marker range of the chunk in source row sy + TR sz
    const int *tile_slot;        // [tile] -> tile slot
    const unsigned *tile_mask;   // [tile slot]
    const int4 *tile_ohdr;       // [position, longest tile first] (tile slot, reach mask, tile id, markers)
    const int2 *tile_orec;       // [position][TR*TR] chunk ranges
    const int *tile_id;          // [tile slot] -> tile
    const int *tile_order;       // tiles, longest first
    const int *n_tiles;
    int tile_cap;
    // collect plan of the marker set (k_collect_plan): where every footprint element goes, and per active cell
    // the run of elements it adds up
    int *fdst;                   // [tile][(TR+3)^2 * ent] -> index into F, or -1 (no cell consumes the element)
    int2 *cell_run;              // [active cell k] (first element in F, number of elements)
    int *n_felem;                // elements handed out so far (plan construction)
    // markers in sorted order
    const float4 *fs;            // (fx, fy, fz, s)
    const float4 *uk;            // u_k
    float4 *du;                  // Delta u, w = cell x index
    // fields
    float4 *U, *G;
    float4 *F;                   // footprint elements, grouped by the cell that consumes them
    const int *cells;            // active-cell list
    const int *n_cells;
};

inline size_t mdf_warp_smem(int tr, const ChunkGeom &cg)
{
    const size_t tf = (size_t)tr + 3;
    const size_t win = (tf * tf * (size_t)cg.ent * 16 + 127) / 128 * 128;
    const size_t foot = (tf * tf * (size_t)cg.ent * 12 + 127) / 128 * 128;
    return win + foot + MDF_STAGE_BYTES;
}

__device__ __forceinline__ int mod_wrap(int i, int n)
{
    i %= n;
    return i < 0 ? i + n : i;
}

__device__ __forceinline__ void cp_async16_cg(void *smem_dst, const void *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// What a warp needs to know about a tile before it touches the tile's markers.
struct TileHdr {
    int t;               // tile id, < 0: none
    int2 rec;            // lane r < TR*TR: sorted-marker range of the chunk in source row r
    int cnt, incl;       // lane r: markers of row r, inclusive prefix over the rows
    int total;           // markers of the tile
    int x0, ty, tz;      // first x cell of the block, tile coordinates in y and z
    unsigned m;          // reach mask: x entries (bits 0..13) | y rows (14..20) | z rows (21..27)
};

template <int TR>
struct TileDims {
    static constexpr int NR = TR * TR, TF = TR + 3, NROWS = TF * TF;
    static constexpr int NRP = NR <= 1 ? 1 : (NR <= 4 ? 4 : 16);     // rows rounded up to a power of two (prefix / search)
    static constexpr int KZ = (TF + 1) / 2;
};

// the shared-memory areas a tile is processed in
struct TileSmem {
    float4 *win;         // [NROWS][ent] window of U^m (w unused)
    float *foot;         // [NROWS][ent][3] footprint
    float4 *sv;          // staging: value + tag of 32 markers (+ 1 padding record)
    float4 *swx;         // staging: x weights
    float *swyz;         // staging: y-z weights [16][33] (weight index major: conflict-free stores by marker, loads by weight)
};

__device__ __forceinline__ size_t tile_win_bytes(int nrows, int ent) { return ((size_t)nrows * ent * 16 + 127) / 128 * 128; }
__device__ __forceinline__ size_t tile_foot_bytes(int nrows, int ent) { return ((size_t)nrows * ent * 12 + 127) / 128 * 128; }

__device__ __forceinline__ TileSmem stage_at(float4 *win, float *foot, char *stage)
{
    TileSmem s;
    s.win = win; s.foot = foot;
    s.sv = reinterpret_cast<float4 *>(stage);
    s.swx = s.sv + MDF_STAGE_RECS;
    s.swyz = reinterpret_cast<float *>(s.swx + MDF_STAGE_RECS);
    return s;
}

// ---- tile header: chunk ranges, their inclusive prefix, geometry (one round trip: all indexed by the position) ----
template <int TR>
__device__ __forceinline__ void tile_load_hdr(const MdfArgs &a, const int pos, const int lane, TileHdr &H)
{
    using D = TileDims<TR>;
    constexpr unsigned FULL = 0xffffffffu;
    H.t = -1;
    H.rec = make_int2(0, 0);
    H.total = 0;
    if (pos < 0) return;
    if (lane < D::NR) H.rec = __ldg(a.tile_orec + (size_t)pos * D::NR + lane);
    const int4 hd = __ldg(a.tile_ohdr + pos);
    const int ts = hd.x;
    H.m = (unsigned)hd.y;
    H.t = hd.z;
    H.cnt = H.rec.y - H.rec.x;
    H.incl = H.cnt;
#pragma unroll
    for (int o = 1; o < D::NRP; o <<= 1) {
        const int v = __shfl_up_sync(FULL, H.incl, o);
        if (lane >= o) H.incl += v;
    }
    H.total = __shfl_sync(FULL, H.incl, D::NRP - 1);
    const int blk = ts % a.cg.nbx, tyz = ts / a.cg.nbx;
    H.ty = tyz % a.tg.nty; H.tz = tyz / a.tg.nty;
    H.x0 = blk * CHUNK_W;
}

// ---- stage the window of U^m: asynchronous 16-byte copies, half a warp per row ------------------------------
// Rows: fy = 0 .. TF-1 (unrolled; with two warps on a tile, `part` takes the rows fy = part, part + nparts, ...),
// fz = 2 k + h.  Row coordinates ty TR - 1 + fy lie in [-1, ny + 4], so one conditional wrap is enough for
// ny >= 4; rows outside a wall axis are never in the mask product.
template <int TR>
__device__ __forceinline__ void tile_issue_window(const MdfArgs &a, const TileHdr &H, float4 *win, const int lane,
                                                  const int part, const int nparts)
{
    using D = TileDims<TR>;
    const int ent = a.cg.ent;
    const int l = lane & 15, h = lane >> 4;
    const unsigned my = H.m >> 14, mz = H.m >> (21 + h);         // bit fy / bit 2 k: the row is reachable
    const bool ex = l < ent && ((H.m >> l) & 1u);                // this lane's window entry is reachable
    const int x = mod_wrap(H.x0 - 1 + l, a.g.nx);
    int zoff[D::KZ];
#pragma unroll
    for (int k = 0; k < D::KZ; ++k) {
        int z = H.tz * TR - 1 + 2 * k + h;
        if (a.g.wallz) z = min(max(z, 0), a.g.nz - 1); else { if (z < 0) z += a.g.nz; else if (z >= a.g.nz) z -= a.g.nz; }
        zoff[k] = z * a.g.ny;
    }
#pragma unroll
    for (int fy = 0; fy < D::TF; ++fy) {
        if (nparts > 1 && (fy % nparts) != part) continue;
        int y = H.ty * TR - 1 + fy;
        if (a.g.wally) y = min(max(y, 0), a.g.ny - 1); else { if (y < 0) y += a.g.ny; else if (y >= a.g.ny) y -= a.g.ny; }
#pragma unroll
        for (int k = 0; k < D::KZ; ++k) {
            if (2 * k + 1 >= D::TF && h) continue;               // fz = 2 k + h < TF
            if (ex && ((my >> fy) & (mz >> (2 * k)) & 1u))
                cp_async16_cg(win + (fy * D::TF + 2 * k + h) * ent + l, a.U + (size_t)(zoff[k] + y) * a.g.nx + x);
        }
    }
}

// the markers of one batch: (source row, sorted index) of this lane's marker, its data in registers
struct MarkerRegs { float4 fs, uk, du; int r, i; };

template <int TR>
__device__ __forceinline__ void tile_fetch(const MdfArgs &a, const TileHdr &H, const int base, const int lane, MarkerRegs &pf)
{
    using D = TileDims<TR>;
    constexpr unsigned FULL = 0xffffffffu;
    const int j = base + lane;
    int r = 0;
#pragma unroll
    for (int step = D::NRP / 2; step >= 1; step >>= 1) {     // the first r with incl[r] > j
        const int v = __shfl_sync(FULL, H.incl, r + step - 1);
        if (j >= v) r += step;
    }
    const int r_first = __shfl_sync(FULL, H.rec.x, r);
    const int r_incl = __shfl_sync(FULL, H.incl, r), r_cnt = __shfl_sync(FULL, H.cnt, r);
    pf.r = r;
    pf.i = r_first + (j - (r_incl - r_cnt));
    if (j < H.total) {
        pf.fs = __ldg(a.fs + pf.i);
        pf.uk = __ldg(a.uk + pf.i);
        pf.du = __ldcg(a.du + pf.i);
    }
}

// ---- phase 1, lane = marker: interpolate, correct, stage the sweep record.
// Returns the marker's tag (source row << 8) | window entry of cell cx - 1.
template <int TR>
__device__ __forceinline__ int tile_phase1(const MdfArgs &a, const TileHdr &H, const MarkerRegs &cur, const bool last,
                                           const TileSmem &sm, const int lane)
{
    using D = TileDims<TR>;
    const int ent = a.cg.ent;
    const float4 fs = cur.fs, uk = cur.uk;
    float4 d = cur.du;
    const int e0 = __float_as_int(d.w) - H.x0;               // window entry of cell cx - 1
    const int sy = cur.r % TR, sz = cur.r / TR;
    float wx[4], wy[4], wz[4];
    peskin4(fs.x, wx);
    peskin4(fs.y, wy);
    peskin4(fs.z, wz);
    const float4 *w0 = sm.win + (sy * D::TF + sz) * ent + e0;
    float ux = 0.f, uy = 0.f, uz = 0.f;
    float *my_wyz = sm.swyz + lane;                  // [ky*4 + kz][marker]
#pragma unroll
    for (int ky = 0; ky < 4; ++ky) {
        float wyz[4];
#pragma unroll
        for (int kz = 0; kz < 4; ++kz) {
            wyz[kz] = wy[ky] * wz[kz];
            const float4 *rowp = w0 + (ky * D::TF + kz) * ent;
            const float4 c0 = rowp[0], c1 = rowp[1], c2 = rowp[2], c3 = rowp[3];
            const float tx = fmaf(wx[3], c3.x, fmaf(wx[2], c2.x, fmaf(wx[1], c1.x, wx[0] * c0.x)));
            const float ty_ = fmaf(wx[3], c3.y, fmaf(wx[2], c2.y, fmaf(wx[1], c1.y, wx[0] * c0.y)));
            const float tz_ = fmaf(wx[3], c3.z, fmaf(wx[2], c2.z, fmaf(wx[1], c1.z, wx[0] * c0.z)));
            ux = fmaf(wyz[kz], tx, ux);
            uy = fmaf(wyz[kz], ty_, uy);
            uz = fmaf(wyz[kz], tz_, uz);
        }
#pragma unroll
        for (int kz = 0; kz < 4; ++kz) my_wyz[(ky * 4 + kz) * MDF_STAGE_RECS] = wyz[kz];
    }
    const float gx = uk.x - ux, gy = uk.y - uy, gz = uk.z - uz;
    d.x = fmaf(fs.w, gx, d.x);
    d.y = fmaf(fs.w, gy, d.y);
    d.z = fmaf(fs.w, gz, d.z);
    a.du[cur.i] = d;
    const int tag = (cur.r << 8) | e0;
    const float tagf = __int_as_float(tag);
    sm.sv[lane] = last ? make_float4(d.x, d.y, d.z, tagf) : make_float4(fs.w * gx, fs.w * gy, fs.w * gz, tagf);
    sm.swx[lane] = make_float4(wx[0], wx[1], wx[2], wx[3]);
    return tag;
}

// ---- phase 2, lane = (half h of the 4-cell x window, target-row offset (jy, jz)): sweep the nb staged markers in
// sorted order (warp-uniform control flow); the staged record of marker jj + 1 is read while marker jj is
// processed.  chg / rowchg: bit jj set = marker jj starts another cell / another source row.
struct SweepState {
    int started;         // a window is open
    int e;               // its first entry
    float *frow;         // footprint row of this lane for the source row being swept
    Acc3 p, q;           // window cells (e + 2h, e + 2h + 1)
};

__device__ __forceinline__ void sweep_flush(float *frow, int ee, const Acc3 &acc)
{
    float *d = frow + ee * 3;
    d[0] += acc.x; d[1] += acc.y; d[2] += acc.z;
}

template <int TR>
__device__ __forceinline__ void tile_sweep(const TileSmem &sm, const int ent, const int nb, const unsigned chg,
                                           const unsigned rowchg, SweepState &st, const int lane)
{
    using D = TileDims<TR>;
    constexpr unsigned FULL = 0xffffffffu;
    const int l = lane & 15, h = lane >> 4;
    const int jy = l >> 2, jz = l & 3;
    const float2 *sw2 = reinterpret_cast<const float2 *>(sm.swx) + h;
    const float *swz = sm.swyz + l * MDF_STAGE_RECS;
    float4 v = sm.sv[0];
    float2 w = sw2[0];
    float wz_ = swz[0];
    const float4 *pv = sm.sv + 1;                    // record jj + 1 (the last read lands on the padding record)
    const float2 *pw = sw2 + 2;
    const float *pz = swz + 1;
    unsigned cbits = chg, rbits = rowchg;
    Acc3 p = st.p, q = st.q;
    int e = st.e, started = st.started;
    float *frow = st.frow;
#pragma unroll 4
    for (int jj = 0; jj < nb; ++jj, ++pv, pw += 2, ++pz, cbits >>= 1, rbits >>= 1) {
        const float4 vn = *pv;
        const float2 wn = *pw;
        const float wzn = *pz;
        if (cbits & 1u) {                            // the sweep moves on to another cell or another source row
            const int tg_ = __float_as_int(v.w);
            const int en = tg_ & 0xff;
            if (rbits & 1u) {                        // another source row (or the first marker of the tile)
                const int rn = tg_ >> 8;
                if (started) { sweep_flush(frow, e + 2 * h, p); sweep_flush(frow, e + 2 * h + 1, q); }
                frow = sm.foot + (((rn % TR) + jy) * D::TF + ((rn / TR) + jz)) * ent * 3;
                p = Acc3{0.f, 0.f, 0.f}; q = Acc3{0.f, 0.f, 0.f};
                e = en;
                started = 1;
            } else {
#pragma unroll 1
                do {                                 // the leftmost window cell is complete
                    if (h == 0) sweep_flush(frow, e, p);
                    const float tx = __shfl_down_sync(FULL, p.x, 16);
                    const float ty_ = __shfl_down_sync(FULL, p.y, 16);
                    const float tz_ = __shfl_down_sync(FULL, p.z, 16);
                    p = q;
                    q.x = h ? 0.f : tx; q.y = h ? 0.f : ty_; q.z = h ? 0.f : tz_;
                } while (++e < en);
            }
        }
        const float vx = v.x * wz_, vy = v.y * wz_, vz = v.z * wz_;
        p.x = fmaf(w.x, vx, p.x); p.y = fmaf(w.x, vy, p.y); p.z = fmaf(w.x, vz, p.z);
        q.x = fmaf(w.y, vx, q.x); q.y = fmaf(w.y, vy, q.y); q.z = fmaf(w.y, vz, q.z);
        v = vn; w = wn; wz_ = wzn;
    }
    st.p = p; st.q = q; st.e = e; st.started = started; st.frow = frow;
}

__device__ __forceinline__ void sweep_close(SweepState &st, const int lane)
{
    const int h = lane >> 4;
    if (st.started) { sweep_flush(st.frow, st.e + 2 * h, st.p); sweep_flush(st.frow, st.e + 2 * h + 1, st.q); }
    st.started = 0;
}

// ---- hand every footprint element to the cell that consumes it (plan: fdst): all the destinations first
// (independent loads), then the stores.  With two warps on a tile, `part` takes the rows fy = part, part + nparts, ...
template <int TR>
struct TileDst { int o[TileDims<TR>::TF][TileDims<TR>::KZ]; };

// where this lane's footprint elements go (collect plan), -1 = nowhere
template <int TR>
__device__ __forceinline__ void tile_load_dst(const MdfArgs &a, const TileHdr &H, const int lane, const int part,
                                              const int nparts, TileDst<TR> &d)
{
    using D = TileDims<TR>;
    const int ent = a.cg.ent;
    const int l = lane & 15, h = lane >> 4;
    const unsigned my = H.m >> 14, mz = H.m >> (21 + h);
    const bool ex = l < ent && ((H.m >> l) & 1u);
    const int *__restrict__ dst = a.fdst + (size_t)H.t * (D::NROWS * ent) + l;
#pragma unroll
    for (int fy = 0; fy < D::TF; ++fy)
#pragma unroll
        for (int k = 0; k < D::KZ; ++k) {
            d.o[fy][k] = -1;
            if (nparts > 1 && (fy % nparts) != part) continue;
            if (2 * k + 1 >= D::TF && h) continue;
            if (ex && ((my >> fy) & (mz >> (2 * k)) & 1u)) d.o[fy][k] = __ldg(dst + (fy * D::TF + 2 * k + h) * ent);
        }
}

template <int TR>
__device__ __forceinline__ void tile_store(const MdfArgs &a, const float *foot, const int lane, const TileDst<TR> &d)
{
    using D = TileDims<TR>;
    const int ent = a.cg.ent;
    const int l = lane & 15, h = lane >> 4;
#pragma unroll
    for (int fy = 0; fy < D::TF; ++fy)
#pragma unroll
        for (int k = 0; k < D::KZ; ++k)
            if (d.o[fy][k] >= 0) {
                const float *sp = foot + ((fy * D::TF + 2 * k + h) * ent + l) * 3;
                __stcg(a.F + d.o[fy][k], make_float4(sp[0], sp[1], sp[2], 0.f));
            }
}

template <int TR>
__device__ __forceinline__ void tile_writeout(const MdfArgs &a, const TileHdr &H, const float *foot, const int lane,
                                              const int part, const int nparts)
{
    TileDst<TR> d;
    tile_load_dst<TR>(a, H, lane, part, nparts, d);
    tile_store<TR>(a, foot, lane, d);
}

// The tile pass of ONE warp over a stream of tiles (next() hands out positions in the longest-first order, < 0 =
// no more).  Software pipeline across tiles: the warp draws its next tile when it starts on the last 32 markers
// of the current one (late, so that the dynamic balance is kept), and as soon as those are interpolated (the
// window is dead from then on) it requests the next tile's window and first 32 markers, which arrive during
// the last sweep and the write-out of the current tile.  wsm = the warp's shared memory (mdf_warp_smem bytes).
// first tile of a warp's stream, loaded ahead of time: header and the first 32 markers do not depend on U, so the
// persistent kernel requests them BEFORE the grid barrier that ends the previous phase
struct TilePre { TileHdr H; MarkerRegs cur; };

template <int TR, class Next>
__device__ __forceinline__ void mdf_tile_prefetch(const MdfArgs &a, const int lane, TilePre &P, Next &&next)
{
    tile_load_hdr<TR>(a, next(), lane, P.H);
    if (P.H.t >= 0) tile_fetch<TR>(a, P.H, 0, lane, P.cur);
}

template <int TR, class Next>
__device__ __forceinline__ void mdf_tile_loop(const MdfArgs &a, const bool last, char *wsm, const int lane, Next &&next,
                                              const TilePre *pre = nullptr)
{
    using D = TileDims<TR>;
    constexpr unsigned FULL = 0xffffffffu;
    const int ent = a.cg.ent;
    const size_t win_bytes = tile_win_bytes(D::NROWS, ent), foot_bytes = tile_foot_bytes(D::NROWS, ent);
    const TileSmem sm = stage_at(reinterpret_cast<float4 *>(wsm), reinterpret_cast<float *>(wsm + win_bytes),
                                 wsm + win_bytes + foot_bytes);
    TileHdr H, Hn;
    MarkerRegs cur;
    if (pre) {
        H = pre->H; cur = pre->cur;
        if (H.t < 0) return;
        tile_issue_window<TR>(a, H, sm.win, lane, 0, 1);
    } else {
        tile_load_hdr<TR>(a, next(), lane, H);
        if (H.t < 0) return;
        tile_issue_window<TR>(a, H, sm.win, lane, 0, 1);
        tile_fetch<TR>(a, H, 0, lane, cur);
    }

    while (H.t >= 0) {
        const int total = H.total;
        // zero the footprint while the window copies and the first markers are in flight
        {
            float4 *f4 = reinterpret_cast<float4 *>(sm.foot);
            const int n4 = (int)(foot_bytes / 16);
            for (int i = lane; i < n4; i += 32) f4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        cp_async_wait_all();
        __syncwarp();

        // ---- the tile's markers, 32 at a time -------------------------------------------------------------
        // single-row tiles (small marker sets, latency-bound): the destinations are requested now, not after the sweep
        TileDst<TR> dst_early;
        if (TR == 1) tile_load_dst<TR>(a, H, lane, 0, 1, dst_early);
        SweepState st;
        st.started = 0; st.e = 0; st.frow = sm.foot;
        st.p = Acc3{0.f, 0.f, 0.f}; st.q = Acc3{0.f, 0.f, 0.f};
        int tag_cur = -1;                            // tag of the last marker swept, -1 = none yet
        Hn.t = -1;
        if (total <= 0) tile_load_hdr<TR>(a, next(), lane, Hn);
        for (int base = 0; base < total; base += MDF_BATCH) {
            const int nb = min(MDF_BATCH, total - base);
            const bool last_batch = base + MDF_BATCH >= total;
            if (last_batch) tile_load_hdr<TR>(a, next(), lane, Hn);
            int tag = -2;
            if (lane < nb) tag = tile_phase1<TR>(a, H, cur, last, sm, lane);
            // which staged markers start another cell / another source row (warp-uniform bit masks: the sweep
            // branches on registers, not on a value it has just loaded)
            const int prev_tag = __shfl_up_sync(FULL, tag, 1);
            const int before = lane == 0 ? tag_cur : prev_tag;
            const unsigned chg = __ballot_sync(FULL, lane < nb && tag != before);
            const unsigned rowchg = __ballot_sync(FULL, lane < nb && ((tag ^ before) >> 8) != 0);
            tag_cur = __shfl_sync(FULL, tag, nb - 1);
            __syncwarp();                                // staging buffer complete; nobody reads the window any more
            if (!last_batch) {
                tile_fetch<TR>(a, H, base + MDF_BATCH, lane, cur);     // in flight during the sweep
            } else if (Hn.t >= 0) {
                tile_issue_window<TR>(a, Hn, sm.win, lane, 0, 1);      // the window is dead: bring in the next tile's,
                tile_fetch<TR>(a, Hn, 0, lane, cur);                   // and its first markers
            }
            tile_sweep<TR>(sm, ent, nb, chg, rowchg, st, lane);
            __syncwarp();                                // every lane is done with the staging buffer
        }
        sweep_close(st, lane);
        __syncwarp();
        if (TR == 1) tile_store<TR>(a, sm.foot, lane, dst_early);
        else tile_writeout<TR>(a, H, sm.foot, lane, 0, 1);
        __syncwarp();
        H = Hn;
    }
}

// tile pass as a kernel of its own: persistent grid, tiles handed out longest first through a cursor
template <int TR>
__global__ void __launch_bounds__(MDF_WARPS * 32, MDF_MIN_BLOCKS)
k_mdf_tiles(const __grid_constant__ MdfArgs a, int *__restrict__ cursor, int last, int warp_smem)
{
    extern __shared__ __align__(128) char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nt = min(*a.n_tiles, a.tile_cap);
    char *wsm = smem + (size_t)warp * warp_smem;
    mdf_tile_loop<TR>(a, last != 0, wsm, lane, [&]() {
        int t = 0;
        if (lane == 0) { t = atomicAdd(cursor, 1); t = t < nt ? t : -1; }
        return __shfl_sync(0xffffffffu, t, 0);
    });
}

// ---- two warps per tile ---------------------------------------------------------------------------------------
// A block is ONE pair of warps on one tile.  The tile's source rows are cut at the row where the marker count
// reaches half the tile's: warp 0 takes the rows up to it, warp 1 the rest.  The two share the tile's window of U^m
// (read only) and otherwise work on their own: each interpolates and sweeps ITS rows' markers, 32 at a time, into a
// footprint of its own; the write-out adds the two footprints (warp 0's first: the order is fixed) and hands the
// elements to the cells.  No barrier inside the tile, two around it.  Against one warp per tile: the longest tile
// takes half as long (the tail of the pass), and 16 instead of 12 warps fit on an SM (28 KB per pair at TR = 4).
inline size_t mdf_pair_smem(int tr, const ChunkGeom &cg)
{
    const size_t tf = (size_t)tr + 3;
    const size_t win = (tf * tf * (size_t)cg.ent * 16 + 127) / 128 * 128;
    const size_t foot = (tf * tf * (size_t)cg.ent * 12 + 127) / 128 * 128;
    return win + 2 * (foot + MDF_STAGE_BYTES);
}

#ifndef MDF_PAIR_MIN_BLOCKS_CFG
#define MDF_PAIR_MIN_BLOCKS_CFG 8
#endif

// footprint elements of the rows fy = part, part + 2, ...: the sum of the two warps' footprints goes to the cells
template <int TR>
__device__ __forceinline__ void pair_writeout(const MdfArgs &a, const TileHdr &H, const float *foot0, const float *foot1,
                                              const int lane, const int part)
{
    using D = TileDims<TR>;
    const int ent = a.cg.ent;
    const int l = lane & 15, h = lane >> 4;
    TileDst<TR> d;
    tile_load_dst<TR>(a, H, lane, part, 2, d);
#pragma unroll
    for (int fy = 0; fy < D::TF; ++fy)
#pragma unroll
        for (int k = 0; k < D::KZ; ++k)
            if (d.o[fy][k] >= 0) {
                const int off = ((fy * D::TF + 2 * k + h) * ent + l) * 3;
                __stcg(a.F + d.o[fy][k], make_float4(foot0[off] + foot1[off], foot0[off + 1] + foot1[off + 1],
                                                      foot0[off + 2] + foot1[off + 2], 0.f));
            }
}

template <int TR>
__global__ void __launch_bounds__(64, MDF_PAIR_MIN_BLOCKS_CFG)
k_mdf_pairs(const __grid_constant__ MdfArgs a, int *__restrict__ cursor, int last_i)
{
    using D = TileDims<TR>;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(128) char smem[];
    __shared__ int s_pos[2];
    const bool last = last_i != 0;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int nt = min(*a.n_tiles, a.tile_cap);
    const int ent = a.cg.ent;
    const size_t win_bytes = tile_win_bytes(D::NROWS, ent), foot_bytes = tile_foot_bytes(D::NROWS, ent);
    float *foot0 = reinterpret_cast<float *>(smem + win_bytes);
    float *foot1 = reinterpret_cast<float *>(smem + win_bytes + foot_bytes);
    const TileSmem sm = stage_at(reinterpret_cast<float4 *>(smem), w ? foot1 : foot0,
                                 smem + win_bytes + 2 * foot_bytes + (size_t)w * MDF_STAGE_BYTES);
    if (threadIdx.x == 0) { const int t = atomicAdd(cursor, 1); s_pos[0] = t < nt ? t : -1; }
    __syncthreads();
    for (int it = 0;; ++it) {
        const int pos = s_pos[it & 1];
        if (pos < 0) break;
        // the next tile is drawn now; its position is read after the barriers of this tile
        if (threadIdx.x == 0) { const int t = atomicAdd(cursor, 1); s_pos[(it + 1) & 1] = t < nt ? t : -1; }
        TileHdr H;
        tile_load_hdr<TR>(a, pos, lane, H);
        tile_issue_window<TR>(a, H, sm.win, lane, w, 2);
        // this warp's rows: up to and including the row where the inclusive count reaches half the tile (warp 0),
        // the rows behind it (warp 1); the header keeps only those, with their prefix redone
        {
            const int half = (H.total + 1) >> 1;
            const unsigned ge = __ballot_sync(FULL, lane < D::NR && H.incl >= half);
            const int b = ge ? __ffs(ge) - 1 : D::NR - 1;
            const bool keep = w == 0 ? lane <= b : lane > b;
            if (!keep) { H.rec.y = H.rec.x; H.cnt = 0; }
            H.incl = H.cnt;
#pragma unroll
            for (int o = 1; o < D::NRP; o <<= 1) {
                const int v = __shfl_up_sync(FULL, H.incl, o);
                if (lane >= o) H.incl += v;
            }
            H.total = __shfl_sync(FULL, H.incl, D::NRP - 1);
        }
        const int total = H.total;
        MarkerRegs cur;
        if (total > 0) tile_fetch<TR>(a, H, 0, lane, cur);
        {
            float4 *f4 = reinterpret_cast<float4 *>(sm.foot);
            const int n4 = (int)(foot_bytes / 16);
            for (int i = lane; i < n4; i += 32) f4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        cp_async_wait_all();
        __syncthreads();                                 // the window is complete (both warps' copies)
        SweepState st;
        st.started = 0; st.e = 0; st.frow = sm.foot;
        st.p = Acc3{0.f, 0.f, 0.f}; st.q = Acc3{0.f, 0.f, 0.f};
        int tag_cur = -1;
        for (int base = 0; base < total; base += MDF_BATCH) {
            const int nb = min(MDF_BATCH, total - base);
            int tag = -2;
            if (lane < nb) tag = tile_phase1<TR>(a, H, cur, last, sm, lane);
            const int prev_tag = __shfl_up_sync(FULL, tag, 1);
            const int before = lane == 0 ? tag_cur : prev_tag;
            const unsigned chg = __ballot_sync(FULL, lane < nb && tag != before);
            const unsigned rowchg = __ballot_sync(FULL, lane < nb && ((tag ^ before) >> 8) != 0);
            tag_cur = __shfl_sync(FULL, tag, nb - 1);
            __syncwarp();
            if (base + MDF_BATCH < total) tile_fetch<TR>(a, H, base + MDF_BATCH, lane, cur);   // in flight during the sweep
            tile_sweep<TR>(sm, ent, nb, chg, rowchg, st, lane);
            __syncwarp();
        }
        sweep_close(st, lane);
        __syncthreads();                                 // both footprints are complete, nobody reads the window any more
        pair_writeout<TR>(a, H, foot0, foot1, lane, w);
        __syncthreads();
    }
}

// ---- stage B ---------------------------------------------------------------------------------------
// Candidates along one axis for the cell coordinate X: source coordinate c = X + 1 - j (wrapped, or
// skipped outside a wall axis); tile = c / tile width (blocks in x: chunk_block); footprint coordinate =
// offset of c in its tile + j.  Distinct (tile, coordinate) pairs only.
template <int MAXC>
struct AxisCandT { int t[MAXC], f[MAXC], n; };

template <bool IS_X, int TR, int MAXC>
__device__ __forceinline__ void axis_candidates_t(int X, int n, int wall, int nbx, AxisCandT<MAXC> &a)
{
    a.n = 0;
    int pt = -1, pf = -1;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        int c = X + 1 - j;
        if (wall) { if (c < 0 || c >= n) continue; } else c = wrap(c, n);
        const int t = IS_X ? chunk_block(c, nbx) : c / TR;
        const int f = c - t * (IS_X ? CHUNK_W : TR) + j;
        if (t != pt || f != pf) {
#pragma unroll
            for (int i = 0; i < MAXC; ++i) if (i == a.n) { a.t[i] = t; a.f[i] = f; }
            ++a.n; pt = t; pf = f;
        }
    }
}

// Collect plan, once per time step (binning stage): every active cell finds the footprint elements of the
// tiles that hold it -- the markers that reach cell X sit in the source cells (X+1-jx, y+1-jy, z+1-jz); per
// axis these four coordinates meet one or two tiles (up to four for single-row tiles and tiny lattices) --
// takes a run of that many slots of F and tells each element where to go (fdst).  The order inside a run is
// fixed (z, y, x candidates ascending), so the sum a cell forms is bitwise reproducible although the position of
// its run is not.  fdst of the tiles in use is pre-set to -1 (k_fill_tiles).
template <int TR, int MAXCX, int MAXCYZ>
__global__ void __launch_bounds__(256)
k_collect_plan(const __grid_constant__ MdfArgs a)
{
    constexpr int TF = TR + 3;
    const Geom &g = a.g;
    const int lane = threadIdx.x & 31;
    constexpr int LPC = MAXCYZ;                      // lanes per cell: lane `sub` of a cell takes the z candidate iz = sub
    constexpr int LSH = LPC == 4 ? 2 : 1;
    static_assert(LPC == 2 || LPC == 4, "two or four z candidates");
    const int sub = lane & (LPC - 1), cl = lane >> LSH;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const int nc = *a.n_cells;
    for (int c0 = (tid - lane) >> LSH; c0 < nc; c0 += stride >> LSH) {
        const int k = c0 + cl;
        AxisCandT<MAXCX> ax;
        AxisCandT<MAXCYZ> ay, az;
        ax.n = ay.n = az.n = 0;
        if (k < nc) {
            const int cell = __ldg(a.cells + k);
            const int row = cell / g.nx;
            const int x = cell - row * g.nx;
            const int z = row / g.ny, y = row - z * g.ny;
            axis_candidates_t<true, TR, MAXCX>(x, g.nx, g.wallx, a.cg.nbx, ax);
            axis_candidates_t<false, TR, MAXCYZ>(y, g.ny, g.wally, 0, ay);
            axis_candidates_t<false, TR, MAXCYZ>(z, g.nz, g.wallz, 0, az);
        }
        // this lane's z candidate (none when sub >= az.n); selected without dynamic indexing
        int zt = 0, zf = 0;
        bool zok = false;
#pragma unroll
        for (int iz = 0; iz < MAXCYZ; ++iz) if (iz == sub && iz < az.n) { zt = az.t[iz]; zf = az.f[iz]; zok = true; }
        auto for_each = [&](auto &&f) {
            if (!zok) return;
#pragma unroll
            for (int iy = 0; iy < MAXCYZ; ++iy)
#pragma unroll
                for (int ix = 0; ix < MAXCX; ++ix) {
                    if (iy >= ay.n || ix >= ax.n) continue;
                    const int ts = tile_slot_of(ax.t[ix], ay.t[iy], zt, a.cg, a.tg);
                    const unsigned m = __ldg(a.tile_mask + ts);
                    if (!((m >> ax.f[ix]) & (m >> (14 + ay.f[iy])) & (m >> (21 + zf)) & 1u)) continue;
                    const int id = __ldg(a.tile_id + ts);
                    if (id < 0 || id >= a.tile_cap) continue;
                    f(((size_t)id * (TF * TF) + ay.f[iy] * TF + zf) * a.cg.ent + ax.f[ix]);
                }
        };
        int cnt = 0;
        for_each([&](size_t) { ++cnt; });
        // lanes in order = cells in order, z candidates ascending inside a cell: the inclusive scan over the warp
        // lays the runs out back to back with their elements in (z, y, x) order
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        int base = 0;
        if (lane == 31 && total) base = atomicAdd(a.n_felem, total);
        base = __shfl_sync(0xffffffffu, base, 31);
        int o = base + incl - cnt;
        const int run_len = __shfl_sync(0xffffffffu, incl, lane | (LPC - 1)) - (incl - cnt);   // sub == 0: elements of the cell
        if (k < nc && sub == 0) a.cell_run[k] = make_int2(o, run_len);
        for_each([&](size_t el) { a.fdst[el] = o++; });
    }
}

// fdst of every tile in use := -1 (elements of the mask product that no active cell consumes stay there)
__global__ void __launch_bounds__(256)
k_fill_tiles(int *__restrict__ fdst, const int *__restrict__ n_tiles, int tile_cap, int elems_per_tile)
{
    const size_t n = (size_t)min(*n_tiles, tile_cap) * (size_t)elems_per_tile;
    int4 *d4 = reinterpret_cast<int4 *>(fdst);
    const size_t n4 = n / 4;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x)
        d4[i] = make_int4(-1, -1, -1, -1);
    if (blockIdx.x == 0 && threadIdx.x < (int)(n - 4 * n4)) fdst[4 * n4 + threadIdx.x] = -1;
}

// One active cell adds up its run of footprint elements, in order.
//   last = false:  U^{m+1}(X) = U^m(X) + sum   (R8)      last = true:  G(X) = sum
__device__ __forceinline__ void mdf_collect_run(const MdfArgs &a, const int cell, const int2 run, const bool last)
{
    const float4 *__restrict__ f = a.F + run.x;
    float sx = 0.f, sy = 0.f, sz = 0.f;
    for (int i0 = 0; i0 < run.y; i0 += 8) {
        float4 v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = (i0 + i < run.y) ? __ldcg(f + i0 + i) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int i = 0; i < 8; ++i) { sx += v[i].x; sy += v[i].y; sz += v[i].z; }
    }
    if (last) {
        a.G[cell] = make_float4(sx, sy, sz, 0.f);
    } else {
        float4 u = __ldcg(a.U + cell);
        u.x += sx; u.y += sy; u.z += sz;
        a.U[cell] = u;
    }
}

__device__ __forceinline__ void mdf_collect_cell(const MdfArgs &a, const int k, const bool last)
{
    mdf_collect_run(a, __ldg(a.cells + k), __ldg(a.cell_run + k), last);
}

__global__ void __launch_bounds__(256)
k_mdf_collect(const __grid_constant__ MdfArgs a, int last)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    const int nc = *a.n_cells;
    for (int k = tid; k < nc; k += stride) mdf_collect_cell(a, k, last != 0);
}

// ---- the whole loop as one persistent kernel ---------------------------------------------------------
// Grid-wide barrier on a monotonic counter (re-armed by the set's next preparation).  All blocks of the
// grid are resident (the host sizes the grid from the occupancy query); blocks of other kernels that
// share the SMs always retire, so the barrier cannot dead-lock.
__device__ __forceinline__ void grid_barrier(unsigned *bar, unsigned &target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        target += gridDim.x;
        __threadfence();
        atomicAdd(bar, 1u);
        unsigned v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while (v < target);
        __threadfence();
    }
    __syncthreads();
}

// a4 for one cell of the active list (same arithmetic as k_moments_active)
__device__ __forceinline__ void moments_cell(const float *__restrict__ src, const Geom &g, const PlaneOffsets &po,
                                             const int cell, float4 *__restrict__ U)
{
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

#ifndef MDFP_MINB_CFG
#define MDFP_MINB_CFG 2
#endif
#ifndef MDFP_WARPS_CFG
#define MDFP_WARPS_CFG 8
#endif
constexpr int MDFP_WARPS = MDFP_WARPS_CFG;   // warps per block of the persistent kernel

// What the persistent kernel needs for the stream-collide of the cells inside the stencils (the words pass), which
// it runs itself once G is complete: one launch and one graph dependency fewer at the end of the step.
struct WordsArgs {
    float *dst;
    CollisionConst cc;
    const unsigned *amask;
    const int *words;
    const int *n_words;
    int enabled;
};

template <int TR>
__global__ void __launch_bounds__(MDFP_WARPS * 32, MDFP_MINB_CFG)
k_mdf_persistent(const __grid_constant__ MdfArgs a, const float *__restrict__ src, const __grid_constant__ PlaneOffsets po,
                 int *__restrict__ cursors, unsigned *__restrict__ bar, int mdf_iters, int warp_smem,
                 const __grid_constant__ WordsArgs wa)
{
    extern __shared__ __align__(128) char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    char *wsm = smem + (size_t)warp * warp_smem;
    const int nt = min(*a.n_tiles, a.tile_cap);
    const int nc = *a.n_cells;
    const int gwarp = warp * gridDim.x + blockIdx.x, nwarps = gridDim.x * MDFP_WARPS;   // consecutive tiles go to different SMs
    const bool dealt = nt <= 2 * nwarps;     // few tiles: dealt statically, longest first (no cursor round trips)
    unsigned target = 0u;
    // every block of this grid is resident now: let the stream-collide pass that runs beside the loop start (it is
    // launched as a programmatic dependent, so that it cannot take the SMs before this grid holds its share)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // the first cell this thread collects is the same in every iteration: its index and run stay in registers
    int my_cell = -1;
    int2 my_run = make_int2(0, 0);
    if (tid < nc) { my_cell = __ldg(a.cells + tid); my_run = __ldg(a.cell_run + tid); }
    // a4: rho, U of eq. (1) on the active cells
    if (my_cell >= 0) moments_cell(src, a.g, po, my_cell, a.U);
    for (int k = tid + stride; k < nc; k += stride) moments_cell(src, a.g, po, __ldg(a.cells + k), a.U);
    // header and first markers of this warp's first tile: requested before the barrier, they arrive behind it
    TilePre P;
    int kd = gwarp - nwarps;
    auto next_dealt = [&]() { kd += nwarps; return kd < nt ? kd : -1; };
    int itc = 0;
    auto next_drawn = [&]() {
        int t = 0;
        if (lane == 0) { t = atomicAdd(cursors + itc, 1); t = t < nt ? t : -1; }
        return __shfl_sync(0xffffffffu, t, 0);
    };
    if (dealt) mdf_tile_prefetch<TR>(a, lane, P, next_dealt); else mdf_tile_prefetch<TR>(a, lane, P, next_drawn);
    grid_barrier(bar, target);
    for (int it = 0; it < mdf_iters; ++it) {
        const bool last = (it == mdf_iters - 1);
        if (dealt) mdf_tile_loop<TR>(a, last, wsm, lane, next_dealt, &P);
        else mdf_tile_loop<TR>(a, last, wsm, lane, next_drawn, &P);
        grid_barrier(bar, target);
        if (my_cell >= 0) mdf_collect_run(a, my_cell, my_run, last);
        for (int k = tid + stride; k < nc; k += stride) mdf_collect_cell(a, k, last);
        if (!last) {
            // the next iteration's first tile (Delta u of its markers was written by this very thread: program order)
            kd = gwarp - nwarps; itc = it + 1;
            if (dealt) mdf_tile_prefetch<TR>(a, lane, P, next_dealt); else mdf_tile_prefetch<TR>(a, lane, P, next_drawn);
            grid_barrier(bar, target);
        }
    }
    if (!wa.enabled) return;
    // a8 on the cells inside the stencils: needs the complete G of every active cell
    grid_barrier(bar, target);
    stream_collide_words(src, wa.dst, a.g, wa.cc, po, wa.amask, wa.words, *wa.n_words, a.G, gwarp, nwarps, lane);
}

}  // namespace lbmk
