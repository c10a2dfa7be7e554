// fdemri_sum.cuh -- S3 + S4: the output-tiled harmonic sum (the hot loop).
//
// Each CTA owns a tile of FDEMRI_TILE consecutive bins of one batch item (one bin per thread, accumulators in
// registers).  It scans the item's strips in their fixed (voice, sign, time) order, turns every strip that
// intersects the tile into "items" -- (voice, sign, segment-branch) with the sub-range of the tile they cover
// and the index of their record -- in shared memory, and every thread whose bin lies in an item's sub-range
// evaluates the term of Eq. 9:
//     A(t) g(X)/sqrt|Fdot| exp{i[2 pi s f t - Phi(t)]},   t = t_k + tau,  F(tau) = s f  (Eq. 6)
// and adds it with the harmonic weights (Eq. 1).  Every bin is written once (S4): no atomics, and the
// summation order of a bin depends only on the data, never on scheduling: results are bitwise reproducible.
// The paper's own layout -- one block per (voice, segment), atomicAdd into global memory (L121) -- is prior art.
#pragma once
#include "fdemri_common.cuh"
#include "airy_tables.inc"

#define FDEMRI_LCAP (3 * FDEMRI_TILE)     // items per round: each candidate strip emits at most 3

struct SumArgs {
    FdemriDims d;
    const double* rec;        // [B][V][S][R_DOUBLES]
    const int2* ent;          // [B][V][2][ent_max]
    const int4* dense;        // [B][dense_cap]
    const int* n_dense;       // [B]
    const int2* bin_range;    // [B] {first, last} bin covered by any strip
    int dense_cap;
    const double4* wts;       // [n_angles][V]
    int n_angles;
    double* hp;               // [B][n_freq][2]
    double* hx;
    unsigned int* tile_counter;
    unsigned long long* stats;
    int total_tiles;
};

// constants as c[][] operands (no immediate materialisation in the loop)
// sin(pi r/2) = r * sum_k S_k r^2k,  cos(pi r/2) = sum_k C_k r^2k,  |r| <= 1/2: truncation 5e-17 / 2e-18
__constant__ double c_sinq[8] = {1.5707963267948966192, -0.64596409750624625366, 0.079692626246167045121,
                                 -0.0046817541353186881007, 0.00016044118478735982187, -3.5988432352120853405e-6,
                                 5.6921729219679268118e-8, -6.6880351098114672325e-10};
__constant__ double c_cosq[9] = {1.0, -1.2337005501361698274, 0.25366950790104801364, -0.020863480763352960873,
                                 0.00091926027483942658024, -0.000025202042373060605481, 4.7108747788181715037e-7,
                                 -6.3866030837918522411e-9, 6.5659631149794723622e-11};
// asymptotic series of g(X) e^{+i pi/4 sgn X} = sum_k i^k a_k u^k, u = 1/X, a_k = prod_j (4/9-(2j-1)^2)/(k! 8^k)
__constant__ double c_gre[7] = {1.0, -0.037133487654320986, 0.05764919041266972, -0.2915913992307505,
                                3.079453030173167, -55.62278536591708, 1533.1694320127956};
__constant__ double c_gim[6] = {-0.06944444444444445, 0.03799305912780064, -0.11609906402551541,
                                0.8776669695100169, -12.341573332345238, 278.46508077760257};

__device__ __forceinline__ void fdemri_g_series(double u, double& re, double& im) {
    const double u2 = u * u;
    if (fabs(u) <= 2.5e-3) {          // |X| >= 400: through a_4, error < 1.2e-14
        re = fma(u2, fma(u2, c_gre[2], c_gre[1]), c_gre[0]);
        im = u * fma(u2, c_gim[1], c_gim[0]);
    } else {                          // 28 <= |X| < 400: through a_12, error < 2e-15
        double r = c_gre[6];
#pragma unroll
        for (int i = 5; i >= 0; --i) r = fma(r, u2, c_gre[i]);
        re = r;
        double q = c_gim[5];
#pragma unroll
        for (int i = 4; i >= 0; --i) q = fma(q, u2, c_gim[i]);
        im = q * u;
    }
}

// x with its sign bit XORed by `mask` (0 or 0x80000000): one integer op on the high word
__device__ __forceinline__ double fdemri_xorsign(double x, unsigned mask) {
    return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}

// sin(2 pi c), cos(2 pi c) for |c| up to ~1e3 cycles (absolute error ~1e-16 + 2 pi ulp(c))
__device__ __forceinline__ void fdemri_sincos_cycles(double c, double& sn, double& cs) {
    const double q = 4.0 * c;
    const double big = 6755399441055744.0;             // 1.5 * 2^52: adding it rounds to the nearest integer
    const double t = q + big;
    const int k = __double2loint(t);                   // low word of the sum = the integer (two's complement)
    const double r = q - (t - big);                    // in [-1/2, 1/2], exact
    const double r2 = r * r;
    double s = c_sinq[7];
#pragma unroll
    for (int i = 6; i >= 0; --i) s = fma(s, r2, c_sinq[i]);
    s *= r;
    double co = c_cosq[8];
#pragma unroll
    for (int i = 7; i >= 0; --i) co = fma(co, r2, c_cosq[i]);
    // rotate by k quarter turns: swap for odd k, then flip signs
    const bool odd = k & 1;
    const double a = odd ? co : s;
    const double b = odd ? s : co;
    sn = fdemri_xorsign(a, ((unsigned)k & 2u) << 30);
    cs = fdemri_xorsign(b, ((unsigned)(k + 1) & 2u) << 30);
}

// Ai(-y), Bi(-y) for 0 <= y < 12.5 from the piecewise Taylor table
__device__ __forceinline__ void fdemri_airy_neg(double y, double& ai, double& bi) {
    int j = (int)(y * 4.0);
    j = min(max(j, 0), FDEMRI_AIRY_NINT - 1);
    double t = y - (0.25 * j + 0.125);
    const double* ca = fdemri_airy_tab[j][0];
    const double* cb = fdemri_airy_tab[j][1];
    double a = ca[FDEMRI_AIRY_DEG], bq = cb[FDEMRI_AIRY_DEG];
#pragma unroll
    for (int i = FDEMRI_AIRY_DEG - 1; i >= 0; --i) {
        a = fma(a, t, ca[i]);
        bq = fma(bq, t, cb[i]);
    }
    ai = a;
    bi = bq;
}

// 32-byte read-only load (sm_100: one 256-bit LDG)
__device__ __forceinline__ double4 fdemri_ld4(const double4* p) {
    double4 v;
    asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}

__device__ __forceinline__ double fdemri_rsqrt_seed(double a) {      // ~21 good bits (MUFU.RSQ64H)
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    return y;
}
// one Newton step of y ~ a^(-1/2):  y <- y + (y/2)(1 - a y^2)
__device__ __forceinline__ double fdemri_rsqrt_step(double y, double a) {
    const double t = a * y;
    const double e = fma(-t, y, 1.0);
    return fma(0.5 * y, e, y);
}

// Root of the monotone segment cubic  FB tau + FC tau^2 + FD tau^3 = x  and 1/sqrt|Fdot| there, without a division.
// Newton with the reciprocal slope taken as +-y^2, y ~ |F'|^(-1/2) refined alongside (the final y is needed anyway).
__device__ __forceinline__ void fdemri_root_monotone(double x, double FB, double FC, double FD, double q1, double q2,
                                                     double q3, double h, double& tau_out, double& Fd_out,
                                                     double& Fdd_out, double& y_out, unsigned int& bad,
                                                     unsigned int& bad_slow) {
    double tau = x * fma(x, fma(x, q3, q2), q1);                 // seed: stored inverse cubic
    double b2, b1, G, c2, dG, y, r;
    // iteration 0
    b2 = fma(tau, FD, FC); b1 = fma(tau, b2, FB); G = fma(tau, b1, -x);
    c2 = fma(tau, FD, b2); dG = fma(tau, c2, b1);
    y = fdemri_rsqrt_seed(fabs(dG));
    r = copysign(y * y, dG);
    tau = fma(-G, r, tau);
    // iteration 1
    b2 = fma(tau, FD, FC); b1 = fma(tau, b2, FB); G = fma(tau, b1, -x);
    c2 = fma(tau, FD, b2); dG = fma(tau, c2, b1);
    y = fdemri_rsqrt_step(y, fabs(dG));
    r = copysign(y * y, dG);
    tau = fma(-G, r, tau);
    // final evaluation and half step
    b2 = fma(tau, FD, FC); b1 = fma(tau, b2, FB); G = fma(tau, b1, -x);
    c2 = fma(tau, FD, b2); dG = fma(tau, c2, b1);
    double Fdd = 2.0 * fma(tau, FD, c2);
    const double ty = fabs(dG) * y;
    const double ey = fma(-ty, y, 1.0);                          // residual of y before this step
    y = fma(0.5 * y, ey, y);
    r = copysign(y * y, dG);
    double delta = G * r;
    // accept when the neglected second-order term is below rounding: in tau (|delta| <= 3e-8 h) and, more
    // demanding near a turnover just outside the segment, in the slope (|F'' delta| <= 1e-6 |F'|); and the
    // iterate must sit in the segment (the root does, by membership R6); and the reciprocal slope r = y^2 that
    // scaled delta must itself be good (|1 - |F'| y^2| <= 1e-3 before its last refinement)
    const double hh = 0.5 * h;
#ifdef FDEMRI_DBG_SLOW
    if (true) {
#else
    if (!(fabs(ey) <= 1e-3 && fabs(delta) <= 6e-8 * hh && fabs(Fdd * delta) <= 1e-6 * fabs(dG) && fabs(tau - hh) <= 1.000000001 * hh)) {
#endif
        // rare: poor seed or nearly flat slope -- plain safeguarded Newton with a true division
        tau = fmin(fmax(tau, 0.0), h);
        int it = 0;
        for (; it < 60; ++it) {
            b2 = fma(tau, FD, FC); b1 = fma(tau, b2, FB); G = fma(tau, b1, -x);
            c2 = fma(tau, FD, b2); dG = fma(tau, c2, b1);
            delta = G / dG;
            if (fabs(delta) <= 1e-14 * h) break;
            tau = fmin(fmax(tau - delta, 0.0), h);
        }
        if (it == 60) bad |= 8u;
        Fdd = 2.0 * fma(tau, FD, c2);
        y = rsqrt(fabs(dG));
        ++bad_slow;
    }
    tau = tau - delta;
    const double Fd = fma(-delta, Fdd, dG);                      // F'(tau - delta) to first order in delta
    Fdd = fma(-6.0 * FD, delta, Fdd);                            // F''(tau - delta), exact for a cubic (the Airy
                                                                 // form near a turnover needs it to 1e-12)
    {
        // last refinement of y = |F'|^(-1/2); its residual e = 1 - |F'| y^2 tells whether y had converged
        const double aFd = fabs(Fd);
        const double t = aFd * y;
        const double e = fma(-t, y, 1.0);
        y = fma(0.5 * y, e, y);                                  // error after the step: 3/8 e^2
        if (!(fabs(e) <= 2e-7)) y = rsqrt(aFd);                  // rare: the slope moved a lot between iterations
    }
    tau_out = tau; Fd_out = Fd; Fdd_out = Fdd; y_out = y;
}

// One term.  R: the (voice, segment) record (24 doubles, 32-byte aligned); sbit = 0 for s=+1, 0x80000000 for s=-1;
// f the bin frequency; brB: second branch of a turnover segment; w = {w+, wx, m phi/2pi}.
// acc = {Re h+, Im h+, Re hx, Im hx}.  cnt = {airy evaluations, slow Newton, error bits}.
__device__ __forceinline__ void fdemri_term(const double* __restrict__ R, unsigned sbit, double f, int brB,
                                            const double4 w, double acc[4], unsigned int cnt[3]) {
    const double4* R4 = reinterpret_cast<const double4*>(R);
    const double4 rF = fdemri_ld4(R4 + 0);       // FA FB FC FD
    const double4 rP = fdemri_ld4(R4 + 1);       // PC BH BL NC
    const double4 rA = fdemri_ld4(R4 + 2);       // Re A
    const double4 rB = fdemri_ld4(R4 + 3);       // Im A
    const double4 rQ = fdemri_ld4(R4 + 4);       // ND TK Q1 Q2
    const double4 rT = fdemri_ld4(R4 + 5);       // Q3 H TYPE spare
    const double FC = rF.z, FD = rF.w;
    const double h = rT.y;
    const double sf = fdemri_xorsign(f, sbit);
    double tau, Fd, Fdd, y, u;
    bool series;                                   // |X| >= 28: asymptotic series, else Airy form
    if (rT.z == 0.0) {
        fdemri_root_monotone(sf - rF.x, rF.y, FC, FD, rQ.z, rQ.w, rT.x, h, tau, Fd, Fdd, y, cnt[2], cnt[1]);
        const double y2 = y * y;
        const double pq = Fdd * y2;
        u = copysign(0.477464829275686 * pq * pq * y2, Fd);      // 1/X = 3 Fdd^2 / (2 pi Fd^3)
        series = fabs(u) <= 0.03571428571428571;
#ifdef FDEMRI_DBG_AIRYTH
        { const double aFd = fabs(Fd); series = 6.283185307179586 * aFd * aFd * aFd >= 84.0 * Fdd * Fdd; }
#endif
    } else {
        // turnover segment: F(tau) - F_e = z^2 (c2 + FD z), z = tau - tau_e; branch A: z < 0, branch B: z > 0
        const double te = rQ.z, Fe = rQ.w, c2 = rT.x;
        const double Delta = sf - Fe;
        double z = sqrt(fmax(Delta / c2, 0.0));
        if (!brB) z = -z;
        const double tol = 1e-14 * h;
        int it = 0;
        for (; it < 40; ++it) {
            double H = fma(z * z, fma(FD, z, c2), -Delta);
            double dH = z * fma(3.0 * FD, z, 2.0 * c2);
            if (dH == 0.0) break;
            double delta = H / dH;
            z -= delta;
            if (fabs(delta) <= tol) break;
        }
        if (it == 40) cnt[2] |= 8u;
        z = brB ? fmin(fmax(z, 0.0), h - te) : fmax(fmin(z, 0.0), -te);
        tau = te + z;
        Fd = z * fma(3.0 * FD, z, 2.0 * c2);          // exact factorisation, no cancellation near Fdot = 0
        Fdd = fma(6.0 * FD, tau, 2.0 * FC);
        if (Fd == 0.0 && Fdd == 0.0) return;           // R10: no term
        const double aFd = fabs(Fd);
        series = 6.283185307179586 * aFd * aFd * aFd >= 84.0 * Fdd * Fdd;
        y = 0.0; u = 0.0;
        if (series) {
            y = rsqrt(aFd);
            const double y2 = y * y;
            const double pq = Fdd * y2;
            u = copysign(0.477464829275686 * pq * pq * y2, Fd);
        }
    }
    // amplitude (two cubics)
    const double Are = fma(tau, fma(tau, fma(tau, rA.w, rA.z), rA.y), rA.x);
    const double Aim = fma(tau, fma(tau, fma(tau, rB.w, rB.z), rB.y), rB.x);
    // phase in cycles (R9): (s f) t_k exactly as p + e, local cubic in tau, knot phase from the record
    const double tk = rQ.y;
    const double p = __dmul_rn(sf, tk);
    const double e = __fma_rn(sf, tk, -p);
    const double big = 6755399441055744.0;
#ifdef FDEMRI_DBG_RINT
    const double pr = p - rint(p);
#else
    const double pr = p - ((p + big) - big);           // p - rint(p), |p| < 2^51
#endif
    const double wv = (sf - rP.y) - rP.z;
    const double loc = tau * fma(tau, fma(tau, rQ.x, rP.w), wv);
    double cyc = ((pr + e) + (rP.x + w.z)) + loc;
    // g(X)/sqrt|Fdot|
    double Sre, Sim;
    if (series) {
        // the e^{-+ i pi/4} of the standard SPA goes into the phase
        double gr, gi;
        fdemri_g_series(u, gr, gi);
        Sre = gr * y;
        Sim = gi * y;
        cyc -= copysign(0.125, Fd);
    } else {
        // |X| < 28: regular Airy form  e^{-iX} pi kap [Ai(-yy) -+ i Bi(-yy)],  kap = (pi|Fddot|)^(-1/3)
        if (Fd == 0.0 && Fdd == 0.0) return;           // R10 (monotone type with a flat cubic)
        const double sig = (Fd >= 0.0) ? 1.0 : -1.0;
        const double kap = rcbrt(3.141592653589793 * fabs(Fdd));
        const double k2 = kap * kap;
        const double yy = k2 * k2 * 9.869604401089358 * Fd * Fd;
        double ai, bi;
        fdemri_airy_neg(yy, ai, bi);
        const double X = 0.6666666666666666 * sig * yy * sqrt(yy);
        cyc -= X * 0.15915494309189535;
        Sre = 3.141592653589793 * kap * ai;
        Sim = -sig * 3.141592653589793 * kap * bi;
        ++cnt[0];
    }
    double sn, cs;
#ifdef FDEMRI_DBG_SINCOSPI
    sincospi(2.0 * cyc, &sn, &cs);
#else
    fdemri_sincos_cycles(cyc, sn, cs);
#endif
    const double Ere = Sre * cs - Sim * sn, Eim = Sre * sn + Sim * cs;
    const double Tre = Are * Ere - Aim * Eim, Tim = Are * Eim + Aim * Ere;
    // weights (O2): s=+1: h+ += w+ T, hx += i wx T;  s=-1: h+ += w+ conj(T), hx += conj(i wx T)
    acc[0] = fma(w.x, Tre, acc[0]);
    acc[1] = fma(fdemri_xorsign(w.x, sbit), Tim, acc[1]);
    acc[2] = fma(-w.y, Tim, acc[2]);
    acc[3] = fma(fdemri_xorsign(w.y, sbit), Tre, acc[3]);
}

// item in shared memory: x = lo | hi << 16 (tile-relative bins), y = global record index
// ((item * V + voice) * n_seg + segment), z = global weight index, w = sign << 30 | branchB << 31
#ifndef FDEMRI_MINBLOCKS
#define FDEMRI_MINBLOCKS 3
#endif
__global__ void __launch_bounds__(FDEMRI_TILE, FDEMRI_MINBLOCKS) k_tile_sum(SumArgs a) {
    __shared__ int4 s_list[FDEMRI_LCAP];
    __shared__ int s_wsum[FDEMRI_TILE / 32];
    __shared__ int s_tile;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const FdemriDims& d = a.d;
    const int V = d.n_modes;
    unsigned int cnt[3] = {0u, 0u, 0u};          // airy evaluations, slow Newton, error bits
    for (;;) {
        __syncthreads();
        if (tid == 0) s_tile = (int)atomicAdd(a.tile_counter, 1u);
        __syncthreads();
        const int gt = s_tile;
        if (gt >= a.total_tiles) break;
        const int b = gt / d.n_tiles, tile = gt - b * d.n_tiles;
        const int64_t bin0 = (int64_t)tile * FDEMRI_TILE;
        const int64_t bin = bin0 + tid;
        const bool valid = bin < d.n_freq;
        const double f = valid ? fdemri_freq(d, bin) : 0.0;
        const int tile_lo = (int)bin0;
        const int tile_hi = (int)min(bin0 + FDEMRI_TILE - 1, d.n_freq - 1);
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        const int2 br = a.bin_range[b];
        const int nd = (br.y < tile_lo || br.x > tile_hi) ? 0 : a.n_dense[b];
        const int4* dense_b = a.dense + (size_t)b * a.dense_cap;
        const int wbase = (a.n_angles > 1 ? b : 0) * V;
        const int rbase = b * V * d.n_seg;
        for (int base = 0; base < nd; base += FDEMRI_TILE) {
            // ---- candidate strip of this thread ----
            const int c = base + tid;
            int remaining = 0, e_next = 0, e0 = 0, ne = 0, dir = 0, vs = 0, s_lo = 0, s_hi = 0;
            const int2* E = nullptr;
            if (c < nd) {
                const int4 s = dense_b[c];
                if (s.x <= tile_hi && s.y >= tile_lo) {
                    vs = s.z >> 1; dir = s.z & 1;
                    e0 = s.w & 0xffff; ne = s.w >> 16;
                    s_lo = s.x; s_hi = s.y;
                    E = a.ent + ((size_t)b * 2 * V + vs) * d.ent_max + e0;
                    const int clo = max(s.x, tile_lo), chi = min(s.y, tile_hi);
                    // entry holding bin x: dir=1: last e with E[e].x <= x;  dir=0: first e with E[e].x <= x
                    int ea, eb;
                    if (dir) {
                        int lo = 0, hi = ne - 1;
                        while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (E[mid].x <= clo) lo = mid; else hi = mid - 1; }
                        ea = lo;
                        hi = ne - 1;
                        while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (E[mid].x <= chi) lo = mid; else hi = mid - 1; }
                        eb = lo;
                    } else {
                        int lo = 0, hi = ne - 1;
                        while (lo < hi) { int mid = (lo + hi) >> 1; if (E[mid].x <= chi) hi = mid; else lo = mid + 1; }
                        ea = lo;
                        hi = ne - 1;
                        while (lo < hi) { int mid = (lo + hi) >> 1; if (E[mid].x <= clo) hi = mid; else lo = mid + 1; }
                        eb = lo;
                    }
                    e_next = ea;
                    remaining = eb - ea + 1;
                }
            }
            // ---- rounds: every candidate emits up to 3 items per round, in candidate order ----
            for (;;) {
                const int n_emit = min(remaining, 3);
                int incl = n_emit;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    int t = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += t;
                }
                if (lane == 31) s_wsum[wid] = incl;
                __syncthreads();
                int woff = 0, total = 0;
#pragma unroll
                for (int i = 0; i < FDEMRI_TILE / 32; ++i) {
                    int ci = s_wsum[i];
                    if (i < wid) woff += ci;
                    total += ci;
                }
                if (total == 0) { __syncthreads(); break; }
                int off = woff + incl - n_emit;
                for (int i = 0; i < n_emit; ++i) {
                    const int e = e_next + i;
                    const int2 en = E[e];
                    int lo_e = en.x, hi_e;
                    if (dir) hi_e = (e + 1 < ne) ? E[e + 1].x - 1 : s_hi;
                    else hi_e = (e > 0) ? E[e - 1].x - 1 : s_hi;
                    lo_e = max(max(lo_e, s_lo), tile_lo) - tile_lo;
                    hi_e = min(min(hi_e, s_hi), tile_hi) - tile_lo;
                    const int seg = en.y & 0x3fffffff;
                    const int v = vs >> 1;
                    s_list[off + i] = make_int4(lo_e | (hi_e << 16), rbase + v * d.n_seg + seg, wbase + v,
                                                ((vs & 1) << 30) | (((en.y >> 30) & 1) << 31));
                }
                e_next += n_emit;
                remaining -= n_emit;
                __syncthreads();
                // ---- evaluate ----
                for (int j = 0; j < total; ++j) {
                    const int4 it = s_list[j];
                    const int lo = it.x & 0xffff, hi = it.x >> 16;
                    if (tid < lo || tid > hi) continue;
                    const unsigned fl = (unsigned)it.w;
                    fdemri_term(a.rec + (size_t)(unsigned)it.y * R_DOUBLES, (fl & 0x40000000u) << 1, f, (int)(fl >> 31),
                                a.wts[(unsigned)it.z], acc, cnt);
                }
                __syncthreads();
            }
        }
        if (valid) {
            const size_t o = ((size_t)b * d.n_freq + bin) * 2;
            *reinterpret_cast<double2*>(a.hp + o) = make_double2(acc[0], acc[1]);
            *reinterpret_cast<double2*>(a.hx + o) = make_double2(acc[2], acc[3]);
        }
    }
    // counters: one atomic per warp
    for (int o = 16; o; o >>= 1) {
        cnt[0] += __shfl_xor_sync(0xffffffffu, cnt[0], o);
        cnt[1] += __shfl_xor_sync(0xffffffffu, cnt[1], o);
        cnt[2] |= __shfl_xor_sync(0xffffffffu, cnt[2], o);
    }
    if (lane == 0) {
        if (cnt[0]) atomicAdd(a.stats + 4, (unsigned long long)cnt[0]);
        if (cnt[1]) atomicAdd(a.stats + 7, (unsigned long long)cnt[1]);
        if (cnt[2]) atomicOr(a.stats + 5, (unsigned long long)cnt[2]);
    }
}
