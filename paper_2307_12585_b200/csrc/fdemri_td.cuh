// fdemri_td.cuh -- the time-domain voice sum of Eq. 1 / Eq. 2, the signal whose Fourier transform
// the stationary-phase sum approximates.  It shares S1 with the frequency-domain path: the
// amplitude cubics and the phase cubic in cycles of every (voice, segment) record are read as they are.
//
//   h(t) = h+ - i hx = sum_v A_v(t) Y_lm e^{-i Phi_v(t)} + [m > 0] (-1)^(l+k) conj(A_v(t)) Y_l,-m e^{+i Phi_v(t)}
// With the real weights of k_weights (w+ = (y+ + (-1)^l y-)/2, wx = (y+ - (-1)^l y-)/2, Y_l,+-m = y+- e^{+-i m phi}) and
// z = A_v(t) e^{-i (Phi_v(t) - m phi)} this is  h = 2 w+ Re z + 2 i wx Im z,  i.e.  h+ += 2 w+ Re z,  hx += -2 wx Im z
// (also for m = 0, where w+ = wx = y/2).
//
// One thread per sample t_j = t0 + j dt; all voices in list order in that thread (fixed summation order).  The knots are
// shared by the voices, so the segment of a sample is found once; neighbouring samples read the same records (broadcast
// loads).  Samples outside [t_0, t_{N-1}) are 0 (R14).
#pragma once
#include "fdemri_common.cuh"

__global__ void __launch_bounds__(256) k_td_sum(FdemriDims d, const double* __restrict__ rec, const double* __restrict__ t_knots,
                                                const double4* __restrict__ wts, int n_angles,
                                                const unsigned char* __restrict__ mode_mask, long long n_samples, double t0,
                                                double dt, double* __restrict__ hp, double* __restrict__ hx) {
    const int b = blockIdx.y;
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_samples) return;
    const int N = d.n_knots, S = d.n_seg, V = d.n_modes;
    const double* tk = t_knots + (size_t)b * N;
    const double tj = __dadd_rn(t0, __dmul_rn((double)j, dt));
    double sp = 0.0, sx = 0.0;
    if (tj >= tk[0] && tj < tk[N - 1]) {
        int lo = 0, hi = N - 1;                                    // t_lo <= tj < t_hi
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(tk + mid) <= tj) lo = mid; else hi = mid;
        }
        const int seg = lo;
        const double tau = tj - __ldg(tk + seg);
        const double4* w = wts + (size_t)(n_angles > 1 ? b : 0) * V;
        const unsigned char* mk = mode_mask ? mode_mask + (size_t)b * V : nullptr;
        const double* R0 = rec + ((size_t)b * V * S + seg) * R_DOUBLES;
        for (int v = 0; v < V; ++v) {
            if (mk && !mk[v]) continue;
            const double4* R4 = reinterpret_cast<const double4*>(R0 + (size_t)v * S * R_DOUBLES);
            const double4 ar = fdemri_ld4(R4 + 2), ai = fdemri_ld4(R4 + 3), ph = fdemri_ld4(R4 + 4);      // Re A, Im A, {PC, BH, BL, NC}
            const double nd = __ldg(reinterpret_cast<const double*>(R4 + 5));
            const double4 wv = fdemri_ld4(w + v);
            // Phi'/2pi = -PC + (BH + BL) tau - NC tau^2 - ND tau^3 - m phi/2pi, reduced as it is built (R9)
            const double p = __dmul_rn(ph.y, tau);
            const double e = __fma_rn(ph.y, tau, -p);
            double cyc = (p - rint(p)) + e;
            cyc += fma(tau, ph.z, -(tau * tau) * fma(tau, nd, ph.w)) - ph.x - wv.z;
            double sn, cs;
            fdemri_sincos_quarter(4.0 * cyc, sn, cs);
            const double Are = fma(tau, fma(tau, fma(tau, ar.w, ar.z), ar.y), ar.x);
            const double Aim = fma(tau, fma(tau, fma(tau, ai.w, ai.z), ai.y), ai.x);
            const double zr = Are * cs + Aim * sn, zi = Aim * cs - Are * sn;               // A e^{-i Phi'}
            sp = fma(2.0 * wv.x, zr, sp);
            sx = fma(-2.0 * wv.y, zi, sx);
        }
    }
    hp[(size_t)b * n_samples + j] = sp;
    hx[(size_t)b * n_samples + j] = sx;
}
