// fdemri_common.cuh -- layouts and small device helpers shared by the kernels of libfdemri.
// Product code: nothing here comes from (or is shared with) oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define FDEMRI_MAX_KNOTS 512
#ifndef FDEMRI_CWARPS
#define FDEMRI_CWARPS 15             // consumer (evaluating) warps per CTA of the sum kernel: with the producer warp 16 warps,
                                     // four per SM sub-partition -- the producer shares its sub-partition with three
                                     // consumers, the other three carry four, so its instructions never set the pace
#endif
#define FDEMRI_BPL 2                 // bins per lane: a consumer warp owns 32*FDEMRI_BPL consecutive bins
#define FDEMRI_TILE (FDEMRI_CWARPS * 32 * FDEMRI_BPL)     // bins per tile (960)
#define FDEMRI_BIN_BLOCK 32          // bins per block of the bin-major sum kernel (one CTA at a time)
#define FDEMRI_SUM_THREADS ((FDEMRI_CWARPS + 1) * 32)     // + one producer warp
#define FDEMRI_CHUNK 32              // staged items per ring stage (one per producer lane)
#ifndef FDEMRI_STAGES
#define FDEMRI_STAGES 8              // ring depth
#endif

// ------------------------------------------------------------------------------------------------
// Record of one (voice, segment) in global memory: everything the sum needs about that piece of
// trajectory that depends neither on the sign s nor on the viewing angles.  24 doubles = 192 B.  tau = t - t_k.
// ------------------------------------------------------------------------------------------------
enum {
    R_FA = 0,   // F(tau) = FA + FB tau + FC tau^2 + FD tau^3  (Eq. 6); FA is the knot value F_k (R6)
    R_FB = 1,
    R_FC = 2,
    R_FD = 3,
    R_Q1 = 4,   // normal segment: seed tau0 = x (Q1 + x (Q2 + x Q3)), x = s f - FA
    R_Q2 = 5,   // one interior extremum: Q1 = tau_e, Q2 = F_e;  two (R5): Q1 = tau_e1, Q2 = F_e1, Q3 = tau_e2, SF = F_e2
    R_Q3 = 6,
    R_H = 7,    // segment length h_k
    R_AR = 8,   // Re A coefficients a,b,c,d  (8..11)   (32-byte aligned: written as one double4)
    R_AI = 12,  // Im A coefficients a,b,c,d  (12..15)
    R_PC = 16,  // phase constant in cycles: -frac(Phi_v(t_k)/2pi)
    R_BH = 17,  // b' = b_Phi/2pi as hi + lo
    R_BL = 18,
    R_NC = 19,  // -c_Phi/2pi
    R_ND = 20,  // -d_Phi/2pi
    R_TK = 21,  // t_k
    R_TYPE = 22,// number of interior extrema of F on the segment: 0.0, 1.0 or 2.0
    R_SF = 23,  // type 0: sign (+-1.0) of dF/dtau on the segment;  type 2: F_e2
    R_DOUBLES = 24
};

// ------------------------------------------------------------------------------------------------
// Staged item in shared memory: one (voice, sign, segment-branch) x tile, written by the producer warp of the
// sum kernel from the record, the sign and the harmonic weights.  Phases are in QUARTER cycles.
// 32 doubles = 256 B; consumers read it with broadcast LDS.
// ------------------------------------------------------------------------------------------------
enum {
    S_META = 0, // int2 {lo | hi << 16 (tile-relative bins), flags: 1 = branch of a segment with extrema (slow path),
                // 2 = a second extremum bounds the branch, 4 = sign s}
    S_F32A = 1, // float2 {FB, FC}: single-precision copies for the first iterate of the inversion
    S_NFA = 2,  // -FA
    S_FB = 3,
    S_FC = 4,
    S_FD = 5,
    S_Q1 = 6,   // monotone segment: seed of the inverse (Q1..Q3).  Branch of a segment with extrema: the extremum it
    S_Q2 = 7,   // starts or ends at, {tau_e, F_e, c2 = C + 3 D tau_e}: F - F_e = z^2 (c2 + D z), z = tau - tau_e; its time
    S_Q3 = 8,   // bracket [ta, tb] in S_F32A, S_F32B; a second extremum {tau_e, F_e, c2} in S_F32C, S_FREE, S_TOLH
    S_TOLH = 9, // acceptance threshold of the last Newton correction, 2e-7 h
    S_HH = 10,  // h/2
    S_F32B = 11,// float2 {FD, Q1}
    S_CU = 12,  // 1/X = CU * (F''/2)^2 / |F'|^3,  CU = sign(F') 6/pi
    S_TK4 = 13, // 4 t_k
    S_WC = 14,  // 4 (F_k - b'), b' = b_Phi/2pi (hi + lo): the linear phase coefficient is 4 (s f - b') = 4 x + WC
    S_FREE = 15,
    S_NC4 = 16, // 4 (-c_Phi/2pi)
    S_ND4 = 17, // 4 (-d_Phi/2pi)
    S_PC4 = 18, // 4 (PC + m phi/2pi) - 0.5 sign(F')     (the e^{-+i pi/4} of the standard SPA, L119; the slow
                // path takes the fold out again with the sign of S_CU)
    S_F32C = 19,// float2 {Q2, Q3}
    S_AR = 20,  // 20..23
    S_AI = 24,  // 24..27
    S_WP = 28,  // w+
    S_SWP = 29, // s w+
    S_NWX = 30, // -wx
    S_SWX = 31, // s wx
    S_DOUBLES = 32
};

struct FdemriDims {
    int n_modes, n_batch, n_knots, n_seg;   // n_seg = n_knots - 1
    int ent_max;                            // entry slots per (voice, sign) = 3 * 32 n_groups: key = vs * ent_max + branch * 32 n_groups + segment
    int n_groups;                           // groups of 32 consecutive segments = ceil(n_seg / 32)
    int64_t n_freq;
    int bin_major;                          // 1: the bin-major sum kernel (sparse grids), 0: the tile-major one
    int tile_bins;                          // bins a CTA owns at a time: FDEMRI_TILE (tile-major) or 8, 16, FDEMRI_BIN_BLOCK = 32 (bin-major)
    int n_tiles;                            // tiles (blocks) per batch item = ceil(n_freq / tile_bins)
    double f0, df, inv_df;                  // inv_df = 1 / df: only to guess a bin index, which is then fixed up exactly
    const double* freq;                     // NULL => uniform grid
    const int* lut;                         // explicit grids: bucket table of fdemri_map.cuh (k_freq_lut), else NULL
    int lut_n;                              // its buckets
};

// frequency of bin i: explicit array, or the uniform grid f0 + i*df with a rounded product and a rounded sum
__device__ __forceinline__ double fdemri_freq(const FdemriDims& d, int64_t i) {
    if (d.freq) return __ldg(d.freq + i);
    return __dadd_rn(d.f0, __dmul_rn((double)i, d.df));
}

// ------------------------------------------------------------------------------------------------
// double-double arithmetic (hi + lo, |lo| <= ulp(hi)/2) for the phase path (R9)
// ------------------------------------------------------------------------------------------------
struct dd {
    double hi, lo;
};
__host__ __device__ __forceinline__ dd dd_make(double a) { return dd{a, 0.0}; }
__device__ __forceinline__ dd two_sum(double a, double b) {
    double s = __dadd_rn(a, b);
    double bb = __dadd_rn(s, -a);
    double e = __dadd_rn(__dadd_rn(a, -__dadd_rn(s, -bb)), __dadd_rn(b, -bb));
    return dd{s, e};
}
__device__ __forceinline__ dd quick_two_sum(double a, double b) {   // |a| >= |b|
    double s = __dadd_rn(a, b);
    double e = __dadd_rn(b, -__dadd_rn(s, -a));
    return dd{s, e};
}
__device__ __forceinline__ dd two_prod(double a, double b) {
    double p = __dmul_rn(a, b);
    double e = __fma_rn(a, b, -p);
    return dd{p, e};
}
__device__ __forceinline__ dd dd_add(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    dd t = two_sum(a.lo, b.lo);
    s.lo = __dadd_rn(s.lo, t.hi);
    s = quick_two_sum(s.hi, s.lo);
    s.lo = __dadd_rn(s.lo, t.lo);
    return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_neg(dd a) { return dd{-a.hi, -a.lo}; }
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, dd_neg(b)); }
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
    dd p = two_prod(a.hi, b.hi);
    p.lo = __dadd_rn(p.lo, __dadd_rn(__dmul_rn(a.hi, b.lo), __dmul_rn(a.lo, b.hi)));
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b) {
    dd p = two_prod(a.hi, b);
    p.lo = __dadd_rn(p.lo, __dmul_rn(a.lo, b));
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_div(dd a, dd b) {
    double q1 = __ddiv_rn(a.hi, b.hi);
    dd r = dd_sub(a, dd_mul_d(b, q1));
    double q2 = __ddiv_rn(r.hi, b.hi);
    r = dd_sub(r, dd_mul_d(b, q2));
    double q3 = __ddiv_rn(r.hi, b.hi);
    dd q = quick_two_sum(q1, q2);
    return dd_add(q, dd_make(q3));
}
// fractional part in [-0.5, 0.5] of a double-double
__device__ __forceinline__ double dd_frac(dd a) {
    double r = rint(a.hi);
    dd f = dd_add(dd{__dadd_rn(a.hi, -r), 0.0}, dd{a.lo, 0.0});   // a.hi - r is exact
    double g = __dadd_rn(f.hi, f.lo);
    return __dadd_rn(g, -rint(g));
}

// 1/(2 pi) as a double-double
#define FDEMRI_INV2PI_HI 0.15915494309189535
#define FDEMRI_INV2PI_LO (-9.839338337591243e-18)
