// fdemri_splines.cuh -- S1: not-a-knot cubic splines on the device.
//
// All components of one batch item share the knots, hence one tridiagonal matrix: it is factorised once per
// item (k_spline_factor) and every component only back-substitutes (one thread per component).
// Unknowns are the second derivatives M_k.  The not-a-knot end conditions
//     h_1 M_0 - (h_0+h_1) M_1 + h_0 M_2 = 0   (and its mirror)
// are substituted into rows 1 and N-2, which leaves a tridiagonal system for M_1..M_{N-2}:
//     row 1   : (h0+h1)(h0+2h1) M_1 + (h1^2-h0^2) M_2                         = h1 r_1
//     row k   : h_{k-1} M_{k-1} + 2(h_{k-1}+h_k) M_k + h_k M_{k+1}            = r_k
//     row N-2 : (hP^2-hL^2) M_{N-3} + (hP+hL)(hL+2hP) M_{N-2}                 = hP r_{N-2}   (hP=h_{N-3}, hL=h_{N-2})
// with r_k = 6[(y_{k+1}-y_k)/h_k - (y_k-y_{k-1})/h_{k-1}].
// The four shared components (f_phi, f_r, Phi_phi, Phi_r) are solved in double-double: the phase splines
// carry 1e5..1e7 rad and must be good to 1e-12 rad (R9).  Amplitudes are solved in double.
#pragma once
#include "fdemri_common.cuh"

// per knot k of item b: fac[(b*N + k)*4 + {0,1,2,3}] = {h_k, lower_k, cp_k, inv_den_k} as dd (double2 hi,lo)
struct SplineFac {
    double2 h, lower, cp, inv_den;
};

__device__ __forceinline__ double2 to2(dd a) { return make_double2(a.hi, a.lo); }
__device__ __forceinline__ dd from2(double2 a) { return dd{a.x, a.y}; }

__global__ void k_spline_factor(int B, int N, const double* __restrict__ t, SplineFac* __restrict__ fac,
                                unsigned long long* __restrict__ flags) {
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const double* tb = t + (size_t)b * N;
    SplineFac* fb = fac + (size_t)b * N;
    bool bad = false;
    for (int k = 0; k < N - 1; ++k) {
        dd h = two_sum(tb[k + 1], -tb[k]);
        if (!(h.hi > 0.0) || !isfinite(h.hi)) bad = true;
        fb[k].h = to2(h);
    }
    fb[N - 1].h = make_double2(0.0, 0.0);
    dd cp_prev = dd_make(0.0);
    for (int k = 1; k <= N - 2; ++k) {
        dd hm = from2(fb[k - 1].h), hk = from2(fb[k].h);
        dd lower, diag, upper;
        if (k == 1) {
            lower = dd_make(0.0);
            diag = dd_mul(dd_add(hm, hk), dd_add(hm, dd_mul_d(hk, 2.0)));
            upper = dd_sub(dd_mul(hk, hk), dd_mul(hm, hm));
        } else {
            lower = hm;
            diag = dd_mul_d(dd_add(hm, hk), 2.0);
            upper = hk;
        }
        if (k == N - 2) {
            // hP = h_{N-3} = hm, hL = h_{N-2} = hk
            dd lo2 = dd_sub(dd_mul(hm, hm), dd_mul(hk, hk));
            dd di2 = dd_mul(dd_add(hm, hk), dd_add(hk, dd_mul_d(hm, 2.0)));
            lower = lo2; diag = di2; upper = dd_make(0.0);      // N >= 4, so k = N-2 > 1
        }
        dd den = dd_sub(diag, dd_mul(lower, cp_prev));
        dd inv = dd_div(dd_make(1.0), den);
        dd cp = dd_mul(upper, inv);
        fb[k].lower = to2(lower);
        fb[k].inv_den = to2(inv);
        fb[k].cp = to2(cp);
        cp_prev = cp;
    }
    if (bad) atomicOr(flags, 4ull);
}

// ---- shared components in double-double -------------------------------------------------------------
// y: 4 pointers (f_phi, f_r, Phi_phi, Phi_r), each [B][N].  out_hi/out_lo: [B][4][N-1][4]
template <int MAXN>
__global__ void k_spline_shared(int B, int N, const double* __restrict__ y0, const double* __restrict__ y1,
                                const double* __restrict__ y2, const double* __restrict__ y3,
                                const SplineFac* __restrict__ fac, double* __restrict__ out_hi,
                                double* __restrict__ out_lo, unsigned long long* __restrict__ flags) {
    int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= B * 4) return;
    int b = id >> 2, c = id & 3;
    const double* y = (c == 0 ? y0 : c == 1 ? y1 : c == 2 ? y2 : y3) + (size_t)b * N;
    const SplineFac* fb = fac + (size_t)b * N;
    dd M[MAXN];
    bool bad = false;
    // forward sweep: M[k] holds dp_k
    dd dp_prev = dd_make(0.0);
    for (int k = 1; k <= N - 2; ++k) {
        dd hm = from2(fb[k - 1].h), hk = from2(fb[k].h);
        if (!isfinite(y[k])) bad = true;
        dd s1 = dd_div(two_sum(y[k + 1], -y[k]), hk);
        dd s0 = dd_div(two_sum(y[k], -y[k - 1]), hm);
        dd r = dd_mul_d(dd_sub(s1, s0), 6.0);
        if (k == 1) r = dd_mul(r, hk);                 // row 1 was multiplied by h_1
        else if (k == N - 2) r = dd_mul(r, hm);        // row N-2 by h_{N-3}
        dd dpk = dd_mul(dd_sub(r, dd_mul(from2(fb[k].lower), dp_prev)), from2(fb[k].inv_den));
        M[k] = dpk;
        dp_prev = dpk;
    }
    // back substitution
    for (int k = N - 3; k >= 1; --k) M[k] = dd_sub(M[k], dd_mul(from2(fb[k].cp), M[k + 1]));
    {
        dd h0 = from2(fb[0].h), h1 = from2(fb[1].h);
        M[0] = dd_div(dd_sub(dd_mul(dd_add(h0, h1), M[1]), dd_mul(h0, M[2])), h1);
        dd hP = from2(fb[N - 3].h), hL = from2(fb[N - 2].h);
        M[N - 1] = dd_div(dd_sub(dd_mul(dd_add(hP, hL), M[N - 2]), dd_mul(hL, M[N - 3])), hP);
    }
    size_t base = (((size_t)b * 4 + c) * (N - 1)) * 4;
    for (int k = 0; k < N - 1; ++k) {
        dd hk = from2(fb[k].h);
        dd slope = dd_div(two_sum(y[k + 1], -y[k]), hk);
        dd bb = dd_sub(slope, dd_div(dd_mul(hk, dd_add(dd_mul_d(M[k], 2.0), M[k + 1])), dd_make(6.0)));
        dd cc = dd_mul_d(M[k], 0.5);
        dd d6 = dd_div(dd_sub(M[k + 1], M[k]), dd_mul_d(hk, 6.0));
        out_hi[base + 4 * k + 0] = y[k];
        out_lo[base + 4 * k + 0] = 0.0;
        out_hi[base + 4 * k + 1] = bb.hi;
        out_lo[base + 4 * k + 1] = bb.lo;
        out_hi[base + 4 * k + 2] = cc.hi;
        out_lo[base + 4 * k + 2] = cc.lo;
        out_hi[base + 4 * k + 3] = d6.hi;
        out_lo[base + 4 * k + 3] = d6.lo;
        if (!isfinite(bb.hi) || !isfinite(cc.hi) || !isfinite(d6.hi)) bad = true;
    }
    if (!isfinite(y[0]) || !isfinite(y[N - 1])) bad = true;
    if (bad) atomicOr(flags, 4ull);
}

// ---- amplitudes in double: one thread per (batch item, mode, re/im) -------------------------------
// amp: [B][V][N][2]; rec: [B][V][N-1][R_DOUBLES], fills R_AR.. / R_AI..
template <int MAXN>
__global__ void k_spline_amp(int B, int V, int N, const double* __restrict__ amp, const SplineFac* __restrict__ fac,
                             double* __restrict__ rec, unsigned long long* __restrict__ flags) {
    size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (size_t)B * V * 2) return;
    int c = (int)(id & 1);
    size_t bv = id >> 1;
    int b = (int)(bv / V);
    const double* y = amp + bv * (size_t)N * 2 + c;     // stride 2
    const SplineFac* fb = fac + (size_t)b * N;
    double M[MAXN];
    bool bad = false;
    double dp_prev = 0.0;
    double ykm = y[0], yk = y[2];
    for (int k = 1; k <= N - 2; ++k) {
        double ykp = y[2 * (k + 1)];
        double hm = fb[k - 1].h.x, hk = fb[k].h.x;
        double r = 6.0 * ((ykp - yk) / hk - (yk - ykm) / hm);
        if (k == 1) r *= hk;
        else if (k == N - 2) r *= hm;
        double dpk = (r - fb[k].lower.x * dp_prev) * fb[k].inv_den.x;
        M[k] = dpk;
        dp_prev = dpk;
        ykm = yk;
        yk = ykp;
    }
    for (int k = N - 3; k >= 1; --k) M[k] = M[k] - fb[k].cp.x * M[k + 1];
    {
        double h0 = fb[0].h.x, h1 = fb[1].h.x;
        M[0] = ((h0 + h1) * M[1] - h0 * M[2]) / h1;
        double hP = fb[N - 3].h.x, hL = fb[N - 2].h.x;
        M[N - 1] = ((hP + hL) * M[N - 2] - hL * M[N - 3]) / hP;
    }
    double* r0 = rec + bv * (size_t)(N - 1) * R_DOUBLES + (c ? R_AI : R_AR);
    yk = y[0];
    for (int k = 0; k < N - 1; ++k) {
        double ykp = y[2 * (k + 1)];
        double hk = fb[k].h.x;
        double bb = (ykp - yk) / hk - hk * (2.0 * M[k] + M[k + 1]) / 6.0;
        double cc = 0.5 * M[k];
        double d6 = (M[k + 1] - M[k]) / (6.0 * hk);
        double4 o = make_double4(yk, bb, cc, d6);
        *reinterpret_cast<double4*>(r0 + (size_t)k * R_DOUBLES) = o;
        if (!isfinite(yk) || !isfinite(bb) || !isfinite(cc) || !isfinite(d6)) bad = true;
        yk = ykp;
    }
    if (!isfinite(yk)) bad = true;
    if (bad) atomicOr(flags, 4ull);
}
