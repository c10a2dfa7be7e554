// fdemri_pairs.cuh -- S2c: the balanced work list.  For every tile of d.tile_bins bins (FDEMRI_TILE for the
// tile-major sum kernel, 1 for the bin-major one), the list of entries
// (voice, sign, segment-branch) whose bin interval intersects it, in the fixed order (voice, sign, time).
//
// "the spline segment in which each value of f falls is predetermined before the summation";
// here the predetermined map is per tile: count -> prefix sum -> fill -> sort (k_pair_pass<0>, k_pair_scan,
// k_pair_pass<1>, k_pair_sort).  The fill uses atomic cursors, so
// the order inside a tile is arbitrary until k_pair_sort puts the keys (unique, = entry index) in ascending
// order: the sum kernel then walks every tile in a data-determined order (bitwise reproducible results).
//   key = (voice*2 + sign) * ent_max + e                (32 bits; the batch item is implied by the tile)
// If the pair list does not fit the work space the flag FDEMRI_BAD_LIST_OVERFLOW is raised: fdemri_sum then fills
// its outputs with NaN and fdemri_get_stats returns FDEMRI_ERR_WORKSPACE with the number of pairs needed.
#pragma once
#include "fdemri_common.cuh"

// k_pair_sort: keys per list the shared-memory sorter takes (longer lists are sorted in place in global memory) and
// threads per CTA, for the tile-major lists (hundreds of keys per 768-bin tile) and the per-bin lists of the bin-major
// mode (as many lists as bins: small CTAs with little shared memory, so that many are resident)
#ifndef FDEMRI_SORT_CAP_TILE
#define FDEMRI_SORT_CAP_TILE 8192
#endif
#ifndef FDEMRI_SORT_THREADS_TILE
#define FDEMRI_SORT_THREADS_TILE 256
#endif
#ifndef FDEMRI_SORT_CAP_BIN
#define FDEMRI_SORT_CAP_BIN 2048
#endif
#ifndef FDEMRI_SORT_THREADS_BIN
#define FDEMRI_SORT_THREADS_BIN 64
#endif

// Tiles t0..t1 of one entry, for every lane of a warp: narrow ranges (the rule) are walked by their own lane, wide
// ones -- an entry of a slowly sweeping voice can cover thousands of bins of a sparse grid -- by the whole warp, so
// that no lane holds the others up.  op(key, tile_base, tile) is called once per (entry, tile) pair, with the
// entry's key and tile base (batch item * n_tiles).  All 32 lanes must call this (has = false: no entry).
template <class Op>
__device__ __forceinline__ void fdemri_for_tiles(bool has, int t0, int t1, unsigned key, unsigned long long tile_base, Op op) {
    const int lane = threadIdx.x & 31;
    const bool wide = has && (t1 - t0) >= 16;
    if (has && !wide)
        for (int t = t0; t <= t1; ++t) op(key, tile_base, t);
    __syncwarp();
    unsigned todo = __ballot_sync(0xffffffffu, wide);
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const int a0 = __shfl_sync(0xffffffffu, t0, src), a1 = __shfl_sync(0xffffffffu, t1, src);
        const unsigned k = __shfl_sync(0xffffffffu, key, src);
        const unsigned long long tb = __shfl_sync(0xffffffffu, tile_base, src);
        for (int t = a0 + lane; t <= a1; t += 32) op(k, tb, t);
    }
}

// One thread per (batch item, voice, sign, entry slot).  MODE 0: count the entries of every tile;  MODE 1: fill the
// lists through atomic cursors (k_pair_sort then fixes the order).  blockDim.x % 32 == 0.
template <int MODE>
__global__ void k_pair_pass(FdemriDims d, const int2* __restrict__ ent, int* __restrict__ tile_cnt,
                            const unsigned int* __restrict__ tile_off, int* __restrict__ tile_cur,
                            unsigned int* __restrict__ pairs, unsigned long long cap) {
    const size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t total = (size_t)d.n_batch * d.n_modes * 2 * d.ent_max;
    const size_t per_item = (size_t)2 * d.n_modes * d.ent_max;
    int2 en = make_int2(0, -1);
    if (id < total) en = ent[id];
    const size_t idc = id < total ? id : total - 1;
    const int b = (int)(idc / per_item);
    const unsigned key = (unsigned)(idc - (size_t)b * per_item);
    fdemri_for_tiles(en.y >= en.x, en.x / d.tile_bins, en.y / d.tile_bins, key, (unsigned long long)b * d.n_tiles,
                     [&](unsigned k, unsigned long long tb, int t) {
                         const size_t gt = (size_t)tb + t;
                         if (MODE == 0) {
                             atomicAdd(tile_cnt + gt, 1);
                         } else {
                             const unsigned long long pos = (unsigned long long)tile_off[gt] + (unsigned)atomicAdd(tile_cur + gt, 1);
                             if (pos < cap) pairs[pos] = k;
                         }
                     });
}

// Exclusive prefix sum of cnt[0..n) into off[0..n], off[n] = total.  One CTA (n is a few thousand per waveform).
// Raises FDEMRI_BAD_LIST_OVERFLOW when the total exceeds the capacity of the pair list.
__global__ void __launch_bounds__(1024) k_pair_scan(size_t n, const int* __restrict__ cnt, unsigned int* __restrict__ off,
                                                    unsigned long long cap, unsigned long long* __restrict__ stats) {
    __shared__ unsigned int s_w[32];
    __shared__ unsigned long long s_base;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_base = 0ull;
    __syncthreads();
    for (size_t start = 0; start < n; start += 4096) {
        // four consecutive elements per thread
        const size_t i0 = start + (size_t)tid * 4;
        unsigned int v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = (i0 + k < n) ? (unsigned)cnt[i0 + k] : 0u;
        const unsigned int mine = v[0] + v[1] + v[2] + v[3];
        unsigned int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) s_w[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            unsigned int w = s_w[lane], wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned int t = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += t;
            }
            s_w[lane] = wi - w;                       // exclusive over warps
        }
        __syncthreads();
        const unsigned long long base = s_base;
        unsigned long long run = base + s_w[wid] + (incl - mine);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (i0 + k < n) off[i0 + k] = (unsigned int)(run > 0xffffffffull ? 0xffffffffull : run);
            run += v[k];
        }
        __syncthreads();
        if (tid == 1023) s_base = run;
        __syncthreads();
    }
    if (tid == 0) {
        const unsigned long long tot = s_base;
        off[n] = (unsigned int)(tot > 0xffffffffull ? 0xffffffffull : tot);
        stats[8] = tot;                                // n_pairs
        if (tot > cap || tot > 0xffffffffull) atomicOr(stats + 5, (unsigned long long)FDEMRI_BAD_LIST_OVERFLOW_BIT);
    }
}

// One CTA per tile: ascending bitonic sort of the tile's keys, in shared memory when they fit and in place in
// global memory otherwise.  Network for arbitrary n: every merge starts with a "flip" step (partner i ^ (2k-1))
// followed by "shift" steps (partner i ^ j), all ascending, so keys past the end act as +infinity and are skipped.
__device__ __forceinline__ void fdemri_bitonic(unsigned int* buf, unsigned int n) {
    unsigned int np = 2;
    while (np < n) np <<= 1;
    for (unsigned int k = 1; k < np; k <<= 1) {                     // merge sorted runs of length k into runs of 2k
        for (unsigned int j = k; j > 0; j >>= 1) {
            for (unsigned int i = threadIdx.x; i < (np >> 1); i += blockDim.x) {
                const unsigned int a = ((i & ~(j - 1)) << 1) | (i & (j - 1));       // bit j clear
                const unsigned int bb = (j == k) ? (a ^ ((j << 1) - 1)) : (a + j);    // flip : shift
                if (bb < n) {
                    const unsigned int x = buf[a], y = buf[bb];
                    if (x > y) { buf[a] = y; buf[bb] = x; }
                }
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(256) k_pair_sort(size_t n_tiles_total, const unsigned int* __restrict__ tile_off,
                                                   unsigned int* __restrict__ pairs, unsigned long long cap,
                                                   unsigned int smem_keys) {
    extern __shared__ unsigned int s_key[];
    const size_t gt = blockIdx.x;
    if (gt >= n_tiles_total) return;
    const unsigned int o0 = tile_off[gt], o1 = tile_off[gt + 1];
    const unsigned int n = o1 - o0;
    if (n < 2u || (unsigned long long)o1 > cap) return;
    if (n > smem_keys) {
        fdemri_bitonic(pairs + o0, n);
        return;
    }
    for (unsigned int i = threadIdx.x; i < n; i += blockDim.x) s_key[i] = pairs[o0 + i];
    __syncthreads();
    fdemri_bitonic(s_key, n);
    for (unsigned int i = threadIdx.x; i < n; i += blockDim.x) pairs[o0 + i] = s_key[i];
}
