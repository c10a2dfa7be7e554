// fdemri_select.cuh -- mode selection by power threshold.
//
// "Within each time step of the sparse array, we take |A_lmkn(t)|^2 and sort the individual modes in descending order
// and compute a cumulative summation.  From this sorted array, we check whether the additional power contributed by an
// individual mode falls below the threshold eps related to the total power emitted. ... The selected modes are given by
// the union of all contributing modes across all time steps."
// Reading (R15): a mode contributes at a time step iff its own power is at least eps times the total power of
// all modes at that step.  In the sorted array the contributing modes are a prefix, so no sort is needed on the
// device: one fixed-order reduction per (item, knot) for the total, one pass per (item, mode) for the union.
#pragma once
#include "fdemri_common.cuh"

// total[b][k] = sum_v |A_v(t_k)|^2, summed in a fixed order (the comparison below must not depend on scheduling).
// One CTA of 256 threads per (batch item, knot).  amp: [B][V][N][2].
__global__ void __launch_bounds__(256) k_select_total(int V, int N, const double* __restrict__ amp, double* __restrict__ total) {
    __shared__ double s_p[256];
    const int b = blockIdx.x / N, k = blockIdx.x - b * N, tid = threadIdx.x;
    double p = 0.0;
    for (int v = tid; v < V; v += 256) {
        const double2 a = *reinterpret_cast<const double2*>(amp + (((size_t)b * V + v) * N + k) * 2);
        p += a.x * a.x + a.y * a.y;
    }
    s_p[tid] = p;
    __syncthreads();
    for (int o = 128; o; o >>= 1) {
        if (tid < o) s_p[tid] += s_p[tid + o];
        __syncthreads();
    }
    if (tid == 0) total[blockIdx.x] = s_p[0];
}

// keep[b][v] = 1 iff |A_v(t_k)|^2 >= eps total[b][k] at some knot k;  n_keep[b] counts them.  One thread per (item, mode).
__global__ void k_select_keep(int B, int V, int N, const double* __restrict__ amp, const double* __restrict__ total, double eps,
                              unsigned char* __restrict__ keep, int* __restrict__ n_keep) {
    const size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (size_t)B * V) return;
    const int b = (int)(id / V);
    const double2* a = reinterpret_cast<const double2*>(amp) + id * N;
    const double* t = total + (size_t)b * N;
    bool k1 = false;
    for (int k = 0; k < N; ++k) {
        const double2 x = a[k];
        k1 = k1 || (x.x * x.x + x.y * x.y >= eps * t[k]);
    }
    keep[id] = k1 ? 1 : 0;
    if (k1) atomicAdd(n_keep + b, 1);
}

// ------------------------------------------------------------------------------------------------------------------
// Second reading of L60 (R15 (b), "cumulative cut"): per time step the modes are sorted by power in
// descending order (ties: mode order), the cumulative sum is formed along the sorted array, and the contributing
// modes are the shortest prefix whose cumulative sum reaches (1 - eps) x total, i.e. sorted mode i is kept iff the sum
// of the modes before it is still below (1 - eps) x total.  One CTA per (batch item, time step): bitonic sort of
// (power, mode index) in shared memory, blocked prefix sum, one flag store per kept mode (the union over the time steps
// is the OR of the stores).  Vp = n_modes rounded up to a power of two (at least 1024); shared memory 12 Vp + 8 KB.
// ------------------------------------------------------------------------------------------------------------------
#define FDEMRI_SELECT_MAX_MODES 16384       // 12 x 16384 + 8 KB of shared memory

__device__ __forceinline__ bool fdemri_sel_before(unsigned long long pa, unsigned ia, unsigned long long pb, unsigned ib) {
    return pa > pb || (pa == pb && ia < ib);             // descending power (bit patterns of non-negative doubles), then mode order
}

__global__ void __launch_bounds__(1024) k_select_cumulative(int V, int N, int Vp, const double* __restrict__ amp, double eps,
                                                            unsigned char* __restrict__ keep) {
    extern __shared__ unsigned long long s_sel[];          // keys [Vp] (power bits), then sums [1024] doubles, then idx [Vp]
    unsigned long long* s_key = s_sel;
    double* s_sum = reinterpret_cast<double*>(s_sel + Vp);
    unsigned* s_idx = reinterpret_cast<unsigned*>(s_sel + Vp + 1024);
    const int b = blockIdx.x / N, k = blockIdx.x - b * N, tid = threadIdx.x;
    for (int v = tid; v < Vp; v += 1024) {
        double p = 0.0;
        if (v < V) {
            const double2 a = *reinterpret_cast<const double2*>(amp + (((size_t)b * V + v) * N + k) * 2);
            p = a.x * a.x + a.y * a.y;
            if (!(p >= 0.0)) p = 0.0;                      // NaN amplitudes are reported by fdemri_build_splines
        }
        s_key[v] = (unsigned long long)__double_as_longlong(p);
        s_idx[v] = (v < V) ? (unsigned)v : 0xffffffffu;    // padding sorts last
    }
    __syncthreads();
    for (int kk = 2; kk <= Vp; kk <<= 1) {
        for (int j = kk >> 1; j > 0; j >>= 1) {
            for (int i = tid; i < Vp; i += 1024) {
                const int l = i ^ j;
                if (l > i) {
                    const unsigned long long pa = s_key[i], pb = s_key[l];
                    const unsigned ia = s_idx[i], ib = s_idx[l];
                    const bool up = (i & kk) == 0;         // this sub-sequence in sorted ("before") order, or reversed
                    const bool swap = up ? fdemri_sel_before(pb, ib, pa, ia) : fdemri_sel_before(pa, ia, pb, ib);
                    if (swap) { s_key[i] = pb; s_key[l] = pa; s_idx[i] = ib; s_idx[l] = ia; }
                }
            }
            __syncthreads();
        }
    }
    // cumulative sum along the sorted array: thread t owns the contiguous chunk [t c, (t + 1) c)
    const int c = Vp / 1024;
    double part = 0.0;
    for (int i = tid * c; i < (tid + 1) * c; ++i) part += __longlong_as_double((long long)s_key[i]);
    s_sum[tid] = part;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {                   // inclusive scan of the chunk sums
        const double t = (tid >= o) ? s_sum[tid - o] : 0.0;
        __syncthreads();
        s_sum[tid] += t;
        __syncthreads();
    }
    const double total = s_sum[1023];
    const double target = (1.0 - eps) * total;
    double before = s_sum[tid] - part;                     // sum of the sorted modes before this chunk
    for (int i = tid * c; i < (tid + 1) * c; ++i) {
        const unsigned v = s_idx[i];
        if (v != 0xffffffffu && before < target) keep[(size_t)b * V + v] = 1;
        before += __longlong_as_double((long long)s_key[i]);
    }
}

// n_keep[b] = number of selected modes of item b.  One CTA per item.
__global__ void __launch_bounds__(256) k_select_count(int V, const unsigned char* __restrict__ keep, int* __restrict__ n_keep) {
    __shared__ int s_c[256];
    const int b = blockIdx.x, tid = threadIdx.x;
    int c = 0;
    for (int v = tid; v < V; v += 256) c += keep[(size_t)b * V + v] ? 1 : 0;
    s_c[tid] = c;
    __syncthreads();
    for (int o = 128; o; o >>= 1) {
        if (tid < o) s_c[tid] += s_c[tid + o];
        __syncthreads();
    }
    if (tid == 0) n_keep[b] = s_c[0];
}
