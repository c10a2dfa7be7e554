// fdemri_splines.cuh -- S1: not-a-knot cubic splines on the device.
//
// Unknowns are the second derivatives M_k.  The not-a-knot end conditions
//     h_1 M_0 - (h_0+h_1) M_1 + h_0 M_2 = 0   (and its mirror)
// are substituted into rows 1 and N-2, which leaves a tridiagonal system for M_1..M_{N-2}:
//     row 1   : (h0+h1)(h0+2h1) M_1 + (h1^2-h0^2) M_2                         = h1 r_1
//     row k   : h_{k-1} M_{k-1} + 2(h_{k-1}+h_k) M_k + h_k M_{k+1}            = r_k
//     row N-2 : (hP^2-hL^2) M_{N-3} + (hP+hL)(hL+2hP) M_{N-2}                 = hP r_{N-2}   (hP=h_{N-3}, hL=h_{N-2})
// with r_k = 6[(y_{k+1}-y_k)/h_k - (y_k-y_{k-1})/h_{k-1}].  The system is strictly diagonally dominant.
//
// The paper leaves the solver open; north_star asks for batched solves on the device.  A sequential Thomas
// sweep per component is a chain of ~N dependent divisions, which on this machine is pure latency (the shared
// double-double solve took 0.46 ms of a 4.5 ms step), so the solves use PARALLEL CYCLIC REDUCTION: one thread per
// row, log2(N) steps, in each of which row i eliminates its couplings to rows i-s and i+s
//     alpha = -a_i / b_{i-s},  gamma = -c_i / b_{i+s}
//     a_i <- alpha a_{i-s},  c_i <- gamma c_{i+s},  b_i <- b_i + alpha c_{i-s} + gamma a_{i+s},
//     d_i <- d_i + alpha d_{i-s} + gamma d_{i+s}
// after which M_i = d_i / b_i.  All right-hand sides of a CTA share the matrix work.
//   * k_spline_shared: one CTA per batch item, the four shared components (f_phi, f_r, Phi_phi, Phi_r) in
//     double-double: the phase splines carry 1e5..1e7 rad and must be good to 1e-12 rad (R9); two or four
//     threads per knot (one or two components each), reciprocals instead of divisions inside the reduction levels.
//   * k_spline_amp: one CTA per FDEMRI_AMP_VOICES voices of a batch item (Re and Im of each), in double.
#pragma once
#include "fdemri_common.cuh"

#define FDEMRI_AMP_VOICES 4          // voices (x Re, Im) per CTA of k_spline_amp

__device__ __forceinline__ double2 to2(dd a) { return make_double2(a.hi, a.lo); }
__device__ __forceinline__ dd from2(double2 a) { return dd{a.x, a.y}; }

// ---- shared components in double-double ----------------------------------------------------------------
// One CTA per batch item; NCT threads per row i (knot), each with 4 / NCT of the four components (right-hand
// sides): thread t has row t / NCT and the components t % NCT, t % NCT + NCT, ...  The matrix part of a reduction
// level (alpha, gamma, the new a, b, c and 1/b) is the same arithmetic in the NCT threads of a row -- computed by
// each, written by the first.  No division inside the levels: every row publishes the double-double reciprocal of
// its diagonal (one double division and a Newton step), its neighbours multiply.
// shared memory per row and buffer: a, b, c, 1/b, d0..d3 as double2 (hi, lo) = 8 double2
#define FDEMRI_SH_ROW 8
#define FDEMRI_SIXTH_HI 0.16666666666666666
#define FDEMRI_SIXTH_LO 9.251858538542970e-18

// 1 / b to double-double accuracy: r0 = fl(1 / b.hi), r = r0 + r0 (1 - b r0)
__device__ __forceinline__ dd dd_recip(dd b) {
    const double r0 = __ddiv_rn(1.0, b.hi);
    const dd e = dd_sub(dd_make(1.0), dd_mul_d(b, r0));
    return quick_two_sum(r0, __dmul_rn(r0, e.hi));
}

// y: 4 pointers (f_phi, f_r, Phi_phi, Phi_r), each [B][N].  out_hi/out_lo: [B][4][N-1][4].  blockDim.x >= NCT * N.
// gridDim.y == 2 (general voices, Eq. 1): the CTAs with blockIdx.y == 1 build the splines of the polar pair
// (f_theta, Phi_theta) from z0, z1 into out2_hi/out2_lo, same layout (components 0 and 1 are read, 2 and 3 repeat them).
template <int NCT>
__global__ void k_spline_shared(int N, const double* __restrict__ t, const double* __restrict__ y0,
                                const double* __restrict__ y1, const double* __restrict__ y2,
                                const double* __restrict__ y3, double* __restrict__ out_hi,
                                double* __restrict__ out_lo, unsigned long long* __restrict__ flags,
                                const double* __restrict__ z0, const double* __restrict__ z1,
                                double* __restrict__ out2_hi, double* __restrict__ out2_lo) {
    extern __shared__ double2 s_sh[];                  // [2][N][FDEMRI_SH_ROW] rows, then h[N], 1/h[N] and M[4][N]
    constexpr int CPT = 4 / NCT;                       // components per thread
    const int b = blockIdx.x, i = threadIdx.x / NCT, cc = threadIdx.x % NCT;
    if (blockIdx.y) {
        y0 = z0; y1 = z1; y2 = z0; y3 = z1;
        out_hi = out2_hi; out_lo = out2_lo;
    }
    double2* buf0 = s_sh;
    double2* buf1 = s_sh + (size_t)N * FDEMRI_SH_ROW;
    double2* s_h = s_sh + (size_t)2 * N * FDEMRI_SH_ROW;          // h_k as dd, k = 0..N-2
    double2* s_ih = s_h + N;                                       // 1 / h_k
    double2* s_M = s_ih + N;                                       // [4][N]
    const double* tb = t + (size_t)b * N;
    const double* yc[4] = {y0 + (size_t)b * N, y1 + (size_t)b * N, y2 + (size_t)b * N, y3 + (size_t)b * N};
    bool bad = false;
    if (cc == 0 && i < N - 1) {
        const dd h = two_sum(tb[i + 1], -tb[i]);
        if (!(h.hi > 0.0) || !isfinite(h.hi)) bad = true;
        s_h[i] = to2(h);
        s_ih[i] = to2(dd_recip(h));
    }
    if (i < N) {
#pragma unroll
        for (int q = 0; q < CPT; ++q) if (!isfinite(yc[cc + q * NCT][i])) bad = true;
    }
    __syncthreads();
    const bool row = (i >= 1 && i <= N - 2);
    dd A = dd_make(0.0), Bq = dd_make(1.0), Cq = dd_make(0.0), D[CPT];
#pragma unroll
    for (int q = 0; q < CPT; ++q) D[q] = dd_make(0.0);
    if (row) {
        const dd hm = from2(s_h[i - 1]), hk = from2(s_h[i]);
        if (i == 1) {
            A = dd_make(0.0);
            Bq = dd_mul(dd_add(hm, hk), dd_add(hm, dd_mul_d(hk, 2.0)));
            Cq = dd_sub(dd_mul(hk, hk), dd_mul(hm, hm));
        } else {
            A = hm;
            Bq = dd_mul_d(dd_add(hm, hk), 2.0);
            Cq = hk;
        }
        if (i == N - 2) {                              // hP = h_{N-3} = hm, hL = h_{N-2} = hk   (N >= 4: i > 1)
            A = dd_sub(dd_mul(hm, hm), dd_mul(hk, hk));
            Bq = dd_mul(dd_add(hm, hk), dd_add(hk, dd_mul_d(hm, 2.0)));
            Cq = dd_make(0.0);
        }
        const dd ihm = from2(s_ih[i - 1]), ihk = from2(s_ih[i]);
#pragma unroll
        for (int q = 0; q < CPT; ++q) {
            const double* y = yc[cc + q * NCT];
            const dd s1 = dd_mul(two_sum(y[i + 1], -y[i]), ihk);
            const dd s0 = dd_mul(two_sum(y[i], -y[i - 1]), ihm);
            dd r = dd_mul_d(dd_sub(s1, s0), 6.0);
            if (i == 1) r = dd_mul(r, hk);             // row 1 was multiplied by h_1
            else if (i == N - 2) r = dd_mul(r, hm);    // row N-2 by h_{N-3}
            D[q] = r;
        }
    }
    // ---- parallel cyclic reduction ----
    double2* cur = buf0;
    double2* nxt = buf1;
    dd IB = dd_recip(Bq);
    if (i < N) {
        double2* me = cur + (size_t)i * FDEMRI_SH_ROW;
        if (cc == 0) { me[0] = to2(A); me[1] = to2(Bq); me[2] = to2(Cq); me[3] = to2(IB); }
#pragma unroll
        for (int q = 0; q < CPT; ++q) me[4 + cc + q * NCT] = to2(D[q]);
    }
    __syncthreads();
    for (int s = 1; s < N - 2; s <<= 1) {
        if (row) {
            dd nA = dd_make(0.0), nC = dd_make(0.0), nB = Bq;
            if (i - s >= 1) {
                const double2* m = cur + (size_t)(i - s) * FDEMRI_SH_ROW;
                const dd alpha = dd_neg(dd_mul(A, from2(m[3])));
                nA = dd_mul(alpha, from2(m[0]));
                nB = dd_add(nB, dd_mul(alpha, from2(m[2])));
#pragma unroll
                for (int q = 0; q < CPT; ++q) D[q] = dd_add(D[q], dd_mul(alpha, from2(m[4 + cc + q * NCT])));
            }
            if (i + s <= N - 2) {
                const double2* p = cur + (size_t)(i + s) * FDEMRI_SH_ROW;
                const dd gamma = dd_neg(dd_mul(Cq, from2(p[3])));
                nC = dd_mul(gamma, from2(p[2]));
                nB = dd_add(nB, dd_mul(gamma, from2(p[0])));
#pragma unroll
                for (int q = 0; q < CPT; ++q) D[q] = dd_add(D[q], dd_mul(gamma, from2(p[4 + cc + q * NCT])));
            }
            A = nA; Bq = nB; Cq = nC;
            IB = dd_recip(Bq);
            double2* me = nxt + (size_t)i * FDEMRI_SH_ROW;
            if (cc == 0) { me[0] = to2(A); me[1] = to2(Bq); me[2] = to2(Cq); me[3] = to2(IB); }
#pragma unroll
            for (int q = 0; q < CPT; ++q) me[4 + cc + q * NCT] = to2(D[q]);
        }
        __syncthreads();
        double2* tmp = cur; cur = nxt; nxt = tmp;
    }
    if (row) {
#pragma unroll
        for (int q = 0; q < CPT; ++q) s_M[(size_t)(cc + q * NCT) * N + i] = to2(dd_mul(D[q], IB));
    }
    __syncthreads();
    if (threadIdx.x < 4) {                             // end values from the not-a-knot relations
        const int c = threadIdx.x;
        const dd h0 = from2(s_h[0]), h1 = from2(s_h[1]);
        const dd M1 = from2(s_M[(size_t)c * N + 1]), M2 = from2(s_M[(size_t)c * N + 2]);
        s_M[(size_t)c * N + 0] = to2(dd_mul(dd_sub(dd_mul(dd_add(h0, h1), M1), dd_mul(h0, M2)), from2(s_ih[1])));
        const dd hP = from2(s_h[N - 3]), hL = from2(s_h[N - 2]);
        const dd Ma = from2(s_M[(size_t)c * N + N - 2]), Mb = from2(s_M[(size_t)c * N + N - 3]);
        s_M[(size_t)c * N + N - 1] = to2(dd_mul(dd_sub(dd_mul(dd_add(hP, hL), Ma), dd_mul(hL, Mb)), from2(s_ih[N - 3])));
    }
    __syncthreads();
    if (i < N - 1) {
        const int k = i;
        const dd hk = from2(s_h[k]), ihk = from2(s_ih[k]);
        const dd sixth = dd{FDEMRI_SIXTH_HI, FDEMRI_SIXTH_LO};
#pragma unroll
        for (int q = 0; q < CPT; ++q) {
            const int c = cc + q * NCT;
            const double* y = yc[c];
            const dd Mk = from2(s_M[(size_t)c * N + k]), Mk1 = from2(s_M[(size_t)c * N + k + 1]);
            const dd slope = dd_mul(two_sum(y[k + 1], -y[k]), ihk);
            const dd bb = dd_sub(slope, dd_mul(dd_mul(hk, dd_add(dd_mul_d(Mk, 2.0), Mk1)), sixth));
            const dd c2 = dd_mul_d(Mk, 0.5);
            const dd d6 = dd_mul(dd_mul(dd_sub(Mk1, Mk), ihk), sixth);
            const size_t base = (((size_t)b * 4 + c) * (N - 1) + k) * 4;
            *reinterpret_cast<double4*>(out_hi + base) = make_double4(y[k], bb.hi, c2.hi, d6.hi);
            *reinterpret_cast<double4*>(out_lo + base) = make_double4(0.0, bb.lo, c2.lo, d6.lo);
            if (!isfinite(bb.hi) || !isfinite(c2.hi) || !isfinite(d6.hi)) bad = true;
        }
    }
    if (bad) atomicOr(flags, 4ull);
}

// ---- amplitudes in double ---------------------------------------------------------------------------------
// amp: [B][V][N][2] (re, im); rec: [B][V][N-1][R_DOUBLES], fills R_AR.. and R_AI..  One CTA per
// FDEMRI_AMP_VOICES voices of one batch item, blockDim.x >= N.  grid = B * ceil(V / FDEMRI_AMP_VOICES).
#define FDEMRI_AMP_ROW (3 + 2 * FDEMRI_AMP_VOICES)
__global__ void k_spline_amp(int V, int N, const double* __restrict__ t, const double* __restrict__ amp,
                             double* __restrict__ rec, unsigned long long* __restrict__ flags) {
    extern __shared__ double s_am[];                   // [2][N][FDEMRI_AMP_ROW] rows, h[N], y[G][N][2], M[G][N][2]
    constexpr int G = FDEMRI_AMP_VOICES;
    const int groups = (V + G - 1) / G;
    const int b = blockIdx.x / groups, v0 = (blockIdx.x - b * groups) * G;
    const int nv = min(G, V - v0);
    const int i = threadIdx.x;
    double* buf0 = s_am;
    double* buf1 = s_am + (size_t)N * FDEMRI_AMP_ROW;
    double* s_h = s_am + (size_t)2 * N * FDEMRI_AMP_ROW;
    double2* s_y = reinterpret_cast<double2*>(s_h + N + (N & 1));          // 16-byte aligned
    double2* s_M = s_y + (size_t)G * N;
    const double* tb = t + (size_t)b * N;
    bool bad = false;
    if (i < N - 1) s_h[i] = tb[i + 1] - tb[i];
    if (i < N) {
        for (int g = 0; g < nv; ++g) {
            const double2 y = *reinterpret_cast<const double2*>(amp + (((size_t)b * V + v0 + g) * N + i) * 2);
            if (!isfinite(y.x) || !isfinite(y.y)) bad = true;
            s_y[(size_t)g * N + i] = y;
        }
    }
    __syncthreads();
    const bool row = (i >= 1 && i <= N - 2);
    double A = 0.0, Bq = 1.0, Cq = 0.0, D[2 * G];
#pragma unroll
    for (int c = 0; c < 2 * G; ++c) D[c] = 0.0;
    if (row) {
        const double hm = s_h[i - 1], hk = s_h[i];
        double scale = 1.0;
        if (i == 1) { A = 0.0; Bq = (hm + hk) * (hm + 2.0 * hk); Cq = hk * hk - hm * hm; scale = hk; }
        else { A = hm; Bq = 2.0 * (hm + hk); Cq = hk; }
        if (i == N - 2) { A = hm * hm - hk * hk; Bq = (hm + hk) * (hk + 2.0 * hm); Cq = 0.0; scale = hm; }
        const double ihk = 1.0 / hk, ihm = 1.0 / hm;
#pragma unroll
        for (int g = 0; g < G; ++g) {
            if (g < nv) {
                const double2 ym = s_y[(size_t)g * N + i - 1], yk = s_y[(size_t)g * N + i], yp = s_y[(size_t)g * N + i + 1];
                D[2 * g] = 6.0 * ((yp.x - yk.x) * ihk - (yk.x - ym.x) * ihm) * scale;
                D[2 * g + 1] = 6.0 * ((yp.y - yk.y) * ihk - (yk.y - ym.y) * ihm) * scale;
            }
        }
    }
    double* cur = buf0;
    double* nxt = buf1;
    if (i < N) {
        double* me = cur + (size_t)i * FDEMRI_AMP_ROW;
        me[0] = A; me[1] = Bq; me[2] = Cq;
#pragma unroll
        for (int c = 0; c < 2 * G; ++c) me[3 + c] = D[c];
    }
    __syncthreads();
    for (int s = 1; s < N - 2; s <<= 1) {
        if (row) {
            double nA = 0.0, nC = 0.0, nB = Bq;
            if (i - s >= 1) {
                const double* m = cur + (size_t)(i - s) * FDEMRI_AMP_ROW;
                const double alpha = -A / m[1];
                nA = alpha * m[0];
                nB = fma(alpha, m[2], nB);
#pragma unroll
                for (int c = 0; c < 2 * G; ++c) D[c] = fma(alpha, m[3 + c], D[c]);
            }
            if (i + s <= N - 2) {
                const double* p = cur + (size_t)(i + s) * FDEMRI_AMP_ROW;
                const double gamma = -Cq / p[1];
                nC = gamma * p[2];
                nB = fma(gamma, p[0], nB);
#pragma unroll
                for (int c = 0; c < 2 * G; ++c) D[c] = fma(gamma, p[3 + c], D[c]);
            }
            A = nA; Bq = nB; Cq = nC;
            double* me = nxt + (size_t)i * FDEMRI_AMP_ROW;
            me[0] = A; me[1] = Bq; me[2] = Cq;
#pragma unroll
            for (int c = 0; c < 2 * G; ++c) me[3 + c] = D[c];
        }
        __syncthreads();
        double* tmp = cur; cur = nxt; nxt = tmp;
    }
    if (row) {
        const double ib = 1.0 / Bq;
#pragma unroll
        for (int g = 0; g < G; ++g) s_M[(size_t)g * N + i] = make_double2(D[2 * g] * ib, D[2 * g + 1] * ib);
    }
    __syncthreads();
    if (i < nv) {                                      // end values from the not-a-knot relations
        const int g = i;
        const double h0 = s_h[0], h1 = s_h[1], hP = s_h[N - 3], hL = s_h[N - 2];
        const double2 M1 = s_M[(size_t)g * N + 1], M2 = s_M[(size_t)g * N + 2];
        const double2 Ma = s_M[(size_t)g * N + N - 2], Mb = s_M[(size_t)g * N + N - 3];
        s_M[(size_t)g * N + 0] = make_double2(((h0 + h1) * M1.x - h0 * M2.x) / h1, ((h0 + h1) * M1.y - h0 * M2.y) / h1);
        s_M[(size_t)g * N + N - 1] = make_double2(((hP + hL) * Ma.x - hL * Mb.x) / hP, ((hP + hL) * Ma.y - hL * Mb.y) / hP);
    }
    __syncthreads();
    if (i < N - 1) {
        const int k = i;
        const double hk = s_h[k], ihk = 1.0 / hk;
        for (int g = 0; g < nv; ++g) {
            const double2 yk = s_y[(size_t)g * N + k], yp = s_y[(size_t)g * N + k + 1];
            const double2 Mk = s_M[(size_t)g * N + k], Mp = s_M[(size_t)g * N + k + 1];
            const double4 re = make_double4(yk.x, (yp.x - yk.x) * ihk - hk * (2.0 * Mk.x + Mp.x) / 6.0, 0.5 * Mk.x,
                                            (Mp.x - Mk.x) * ihk / 6.0);
            const double4 im = make_double4(yk.y, (yp.y - yk.y) * ihk - hk * (2.0 * Mk.y + Mp.y) / 6.0, 0.5 * Mk.y,
                                            (Mp.y - Mk.y) * ihk / 6.0);
            double* r0 = rec + (((size_t)b * V + v0 + g) * (N - 1) + k) * R_DOUBLES;
            *reinterpret_cast<double4*>(r0 + R_AR) = re;
            *reinterpret_cast<double4*>(r0 + R_AI) = im;
            if (!isfinite(re.y) || !isfinite(re.z) || !isfinite(re.w) || !isfinite(im.y) || !isfinite(im.z) || !isfinite(im.w))
                bad = true;
        }
    }
    if (bad) atomicOr(flags, 4ull);
}
