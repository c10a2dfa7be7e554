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
