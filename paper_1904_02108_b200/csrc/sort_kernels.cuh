// Marker binning, part 1 (row a3 of SURVEY.md section 8): stable LSD radix sort of (cell key,
// marker index) pairs, 8 bits per pass, hand-written.  The paper only suggests the reordering
// (last sentence); the sort must be stable with ties broken by the original marker index so
// that the permutation is unique (R20).
//
// One pass = three kernels.  The key array is cut into sub-tiles of `ipw` consecutive items, one
// warp per sub-tile:
//   k_radix_hist    per-sub-tile digit histogram  -> hist[digit][tile]
//   k_radix_scan    block d: exclusive scan of row d over the tiles, row total -> total[d]
//   k_radix_scatter per warp: counters = (exclusive scan of total)[d] + hist[d][tile]; items are
//                   taken 32 at a time in order, ranked inside the warp with __match_any_sync
//                   (lane order = original order), and written to their final slot.
// Stability: lanes in order inside a round, rounds in order inside a sub-tile, sub-tiles in order
// through the row scan.
#pragma once
#include <cuda_runtime.h>

namespace lbmk {

constexpr int SORT_BLOCK = 256;             // 8 warps per block
constexpr int SORT_WARPS = SORT_BLOCK / 32;
constexpr int RADIX = 256;

__global__ void __launch_bounds__(SORT_BLOCK)
k_radix_hist(const unsigned *__restrict__ keys, int n, int ipw, int ntiles, int shift, int *__restrict__ hist)
{
    __shared__ int cnt[SORT_WARPS][RADIX];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int tile = blockIdx.x * SORT_WARPS + wib;
    for (int d = lane; d < RADIX; d += 32) cnt[wib][d] = 0;
    __syncwarp();
    if (tile < ntiles) {
        const int beg = tile * ipw;
        const int end = min(n, beg + ipw);
        for (int i = beg + lane; i < end; i += 32) atomicAdd(&cnt[wib][(keys[i] >> shift) & (RADIX - 1)], 1);
        __syncwarp();
        for (int d = lane; d < RADIX; d += 32) hist[(size_t)d * ntiles + tile] = cnt[wib][d];
    }
}

__global__ void __launch_bounds__(SORT_BLOCK)
k_radix_scan(int *__restrict__ hist, int ntiles, int *__restrict__ total)
{
    __shared__ int wsum[SORT_WARPS];
    __shared__ int carry_s;
    int *row = hist + (size_t)blockIdx.x * ntiles;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < ntiles; base += SORT_BLOCK) {
        const int i = base + threadIdx.x;
        const int v = (i < ntiles) ? row[i] : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) wsum[wib] = incl;
        __syncthreads();
        int woff = 0;
        for (int w = 0; w < wib; ++w) woff += wsum[w];
        const int carry = carry_s;
        if (i < ntiles) row[i] = carry + woff + incl - v;
        __syncthreads();
        if (threadIdx.x == SORT_BLOCK - 1) carry_s = carry + woff + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) total[blockIdx.x] = carry_s;
}

// vals_in == nullptr means "identity" (first pass: the value of item i is i).
__global__ void __launch_bounds__(SORT_BLOCK)
k_radix_scatter(const unsigned *__restrict__ keys_in, const int *__restrict__ vals_in, unsigned *__restrict__ keys_out,
                int *__restrict__ vals_out, int n, int ipw, int ntiles, int shift, const int *__restrict__ hist,
                const int *__restrict__ total)
{
    __shared__ int cnt[SORT_WARPS][RADIX];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int tile = blockIdx.x * SORT_WARPS + wib;
    if (tile >= ntiles) return;   // whole warp leaves together

    // exclusive scan of the 256 digit totals: lane holds digits 8*lane .. 8*lane+7
    int t[8], run = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { t[j] = total[lane * 8 + j]; run += t[j]; }
    int incl = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    int base = incl - run;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const int d = lane * 8 + j;
        cnt[wib][d] = base + hist[(size_t)d * ntiles + tile];
        base += t[j];
    }
    __syncwarp();

    const int beg = tile * ipw;
    const int end = min(n, beg + ipw);
    const unsigned lt = (1u << lane) - 1u;
    for (int r = beg; r < end; r += 32) {
        const int i = r + lane;
        const bool valid = i < end;
        const unsigned key = valid ? keys_in[i] : 0u;
        const int val = valid ? (vals_in ? vals_in[i] : i) : 0;
        const unsigned d = valid ? ((key >> shift) & (RADIX - 1)) : 0xffffffffu;
        const unsigned peers = __match_any_sync(0xffffffffu, d);
        const int leader = __ffs(peers) - 1;
        int old = 0;
        if (valid && lane == leader) old = cnt[wib][d];
        __syncwarp();
        if (valid && lane == leader) cnt[wib][d] = old + __popc(peers);
        old = __shfl_sync(0xffffffffu, old, leader);
        __syncwarp();
        if (valid) {
            const int pos = old + __popc(peers & lt);
            keys_out[pos] = key;
            vals_out[pos] = val;
        }
    }
}

// Small marker sets: all passes in ONE kernel of ONE block (16 warps; warp w owns the w-th contiguous stretch of the
// array; 512 threads so that the block finds room on an SM that already holds a block of the persistent MDF kernel).  Per pass: per-warp digit histograms in shared memory, one thread per digit turns them into the warps'
// start offsets (digit-major, warp-minor: the same order as the three-kernel pass), the warps scatter their items
// 32 at a time with the same __match_any_sync ranking; block barriers order the passes (one block: no grid-wide
// synchronisation is needed).  Same result as the three-kernel passes, nine launches fewer for a 24-bit key.
#ifndef SORT_SMALL_BLOCK_CFG
#define SORT_SMALL_BLOCK_CFG 512
#endif
constexpr int SORT_SMALL_BLOCK = SORT_SMALL_BLOCK_CFG;
constexpr int SORT_SMALL_WARPS = SORT_SMALL_BLOCK / 32;
constexpr int SORT_SMALL_MAX = 32768;       // markers up to which the single-block sort is used

__global__ void __launch_bounds__(SORT_SMALL_BLOCK, 2)
k_radix_sort_small(unsigned *keys0, unsigned *keys1, int *vals0, int *vals1, int n, int npasses)
{
    __shared__ int cnt[SORT_SMALL_WARPS][RADIX];
    __shared__ int dsum[RADIX];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int per = ((n + SORT_SMALL_WARPS - 1) / SORT_SMALL_WARPS + 31) & ~31;
    const int beg = min(n, wib * per), end = min(n, beg + per);
    const unsigned lt = (1u << lane) - 1u;
    for (int p = 0; p < npasses; ++p) {
        // plain pointers: a pass reads what the pass before wrote (no read-only data path)
        const unsigned *kin = (p & 1) ? keys1 : keys0;
        unsigned *kout = (p & 1) ? keys0 : keys1;
        const int *vin = p == 0 ? nullptr : ((p & 1) ? vals1 : vals0);
        int *vout = (p & 1) ? vals0 : vals1;
        const int shift = 8 * p;
        for (int d = lane; d < RADIX; d += 32) cnt[wib][d] = 0;
        __syncwarp();
        for (int i = beg + lane; i < end; i += 32) atomicAdd(&cnt[wib][(kin[i] >> shift) & (RADIX - 1)], 1);
        __syncthreads();
        // one thread per digit (in rounds): exclusive prefix of the digit over the warps, digit total
        for (int d = threadIdx.x; d < RADIX; d += SORT_SMALL_BLOCK) {
            int run = 0;
#pragma unroll 4
            for (int w = 0; w < SORT_SMALL_WARPS; ++w) { const int v = cnt[w][d]; cnt[w][d] = run; run += v; }
            dsum[d] = run;
        }
        __syncthreads();
        // warp 0: exclusive scan of the 256 digit totals, lane holds digits 8 lane .. 8 lane + 7
        if (wib == 0) {
            int t[8], run = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) { t[j] = dsum[lane * 8 + j]; run += t[j]; }
            int incl = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += v;
            }
            int base = incl - run;
#pragma unroll
            for (int j = 0; j < 8; ++j) { dsum[lane * 8 + j] = base; base += t[j]; }
        }
        __syncthreads();
        for (int d = threadIdx.x; d < RADIX; d += SORT_SMALL_BLOCK) {
            const int base = dsum[d];
#pragma unroll 4
            for (int w = 0; w < SORT_SMALL_WARPS; ++w) cnt[w][d] += base;
        }
        __syncthreads();
        // the items of round r + 1 are requested while round r is ranked (one warp per stretch: nothing else hides
        // the load latency)
        unsigned key_n = (beg + lane < end) ? kin[beg + lane] : 0u;
        int val_n = (beg + lane < end) ? (vin ? vin[beg + lane] : beg + lane) : 0;
        for (int r = beg; r < end; r += 32) {
            const int i = r + lane;
            const bool valid = i < end;
            const unsigned key = key_n;
            const int val = val_n;
            if (i + 32 < end) { key_n = kin[i + 32]; val_n = vin ? vin[i + 32] : i + 32; }
            const unsigned d = valid ? ((key >> shift) & (RADIX - 1)) : 0xffffffffu;
            const unsigned peers = __match_any_sync(0xffffffffu, d);
            const int leader = __ffs(peers) - 1;
            int old = 0;
            if (valid && lane == leader) old = cnt[wib][d];
            __syncwarp();
            if (valid && lane == leader) cnt[wib][d] = old + __popc(peers);
            old = __shfl_sync(0xffffffffu, old, leader);
            __syncwarp();
            if (valid) {
                const int pos = old + __popc(peers & lt);
                kout[pos] = key;
                vout[pos] = val;
            }
        }
        __syncthreads();                             // the pass's output is complete (and visible) for the whole block
    }
}

}  // namespace lbmk
