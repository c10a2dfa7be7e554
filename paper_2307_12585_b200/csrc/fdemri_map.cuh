// fdemri_map.cuh -- S0 (harmonic weights) and S2 (segment records + segment->bin-range map).
//
// S2 follows PAPER.md L103 (A..D = mode-number-weighted sums of the fundamental-frequency spline
// coefficients) and L105 ("the spline segment in which each value of f falls is predetermined before the
// summation").  The map is inverted with respect to the paper: instead of a segment index per (f, voice) it
// stores, per (voice, sign, segment-branch), the contiguous interval of bins the branch covers ("entry");
// fdemri_pairs.cuh turns the entries into per-tile work lists.
//
// Membership (R6-R8), decided on doubles only: the knot values F_k (fdemri_knotF), the extremum
// value F_e of a turnover segment (record slot R_Q2) and the bin frequencies f_i.
//   branch from value Va (start, in time) to Vb (end):
//     normal segment        : Va = F_k included, Vb = F_{k+1} excluded          (half-open in time, R6)
//     turnover, 1st branch  : Va = F_k included, Vb = F_e included               (R7)
//     turnover, last branch : Va = F_e excluded, Vb = F_{k+1} excluded
//     two extrema (R5), middle branch: Va = F_e1 excluded, Vb = F_e2 included
//   a bin f_i > 0 belongs to the branch for sign s when s*f_i lies between Va and Vb under those rules.
#pragma once
#include "fdemri_common.cuh"

// ------------------------------------------------------------------------------------------------
// S0: weights.  -2Y_lm(theta, phi) = sqrt((2l+1)/4pi) d^l_{m,2}(theta) e^{i m phi}  (Wigner small-d), hence
//   W+ = e^{i m phi} w+,  Wx = i e^{i m phi} wx   with real  w+ = (y+ + (-1)^l y-)/2,  wx = (y+ - (-1)^l y-)/2,
//   y+- = -2Y_{l,+-m}(theta, 0);  m = 0: w+ = wx = y/2 (R1, R2).
// The factor e^{i m phi} goes into the phase as m*phi/2pi cycles.
// ------------------------------------------------------------------------------------------------
// The theta-independent coefficients of the Wigner sum are tabulated per distinct (l, m) on the host at plan time
// (fdemri.cu: build_weight_table), so that a call only evaluates  sum_j C_j ch^(p0-2j) sh^(q0+2j).
__device__ __forceinline__ double fdemri_ipow(double x, int n) {      // x^n, n >= 0, by squaring
    double r = 1.0;
    while (n) {
        if (n & 1) r *= x;
        x *= x;
        n >>= 1;
    }
    return r;
}
__device__ __forceinline__ double fdemri_wigner_sum(const int4 meta, const double* __restrict__ coef, double ch, double sh) {
    // meta = {number of terms, p0, q0, offset of the coefficients}
    const double* c = coef + meta.w;
    double tot = 0.0;
    for (int j = 0; j < meta.x; ++j) {
        // ch^(p0 - 2j) sh^(q0 + 2j) without dividing (ch or sh may vanish): both exponents stay >= 0
        tot = fma(c[j], fdemri_ipow(ch, meta.y - 2 * j) * fdemri_ipow(sh, meta.z + 2 * j), tot);
    }
    return tot;
}

// wts: [n_angles][V] double4 {w+, wx, m*phi/2pi (cycles, reduced), 0}
// kk: polar harmonic k of every voice (general voices, Eq. 1) or NULL: the partner (l,-m,-k,-n) carries (-1)^(l+k) (R16).
__global__ void k_weights(int n_angles, int V, const int* __restrict__ lmn, const int* __restrict__ kk,
                          const int* __restrict__ lm_index,
                          const int4* __restrict__ wmeta, const double* __restrict__ wcoef,
                          const double* __restrict__ angles, double theta0, double phi0, double4* __restrict__ wts,
                          unsigned long long* __restrict__ sum_counters) {
    int id = blockIdx.x * blockDim.x + threadIdx.x;
    // the counters of the sum that follows on the stream: n_airy (slot 4), the tile counter (6), n_slow (7), n_pairs (8),
    // the sum's flags (9) -- cleared here instead of by two memsets in front of every sum
    if (sum_counters && id == 0) {
        sum_counters[4] = 0ull; sum_counters[6] = 0ull; sum_counters[7] = 0ull; sum_counters[8] = 0ull; sum_counters[9] = 0ull;
    }
    if (id >= n_angles * V) return;
    int a = id / V, v = id - a * V;
    const int m = lmn[3 * v + 1];
    const int lm = lm_index[v];
    // one pair of angles for the whole batch travels as kernel arguments (no copy); per-item angles come from `angles`
    double theta = angles ? angles[2 * a] : theta0, phi = angles ? angles[2 * a + 1] : phi0;
    double ch = cos(0.5 * theta), sh = sin(0.5 * theta);
    const double yp = fdemri_wigner_sum(wmeta[2 * lm], wcoef, ch, sh);            // -2Y_{l,m}(theta, 0)
    double wp, wx;
    if (m > 0) {
        double ym = fdemri_wigner_sum(wmeta[2 * lm + 1], wcoef, ch, sh);          // (-1)^l -2Y_{l,-m}(theta, 0)
        if (kk && (kk[v] & 1)) ym = -ym;
        wp = 0.5 * (yp + ym);
        wx = 0.5 * (yp - ym);
    } else {
        wp = 0.5 * yp;
        wx = 0.5 * yp;
    }
    double cyc = (double)m * phi * 0.15915494309189535;
    cyc -= rint(cyc);
    wts[id] = make_double4(wp, wx, cyc, 0.0);
}

// ------------------------------------------------------------------------------------------------
// S2a: records.  One thread per (batch item, voice, segment).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double fdemri_knotF(int m, int n, double fphi, double fr) {
    // knot value of F_v as plainly rounded doubles (R6): products rounded, then the sum rounded
    return __dadd_rn(__dmul_rn((double)m, fphi), __dmul_rn((double)n, fr));
}

__device__ __forceinline__ dd fdemri_combine(int m, int n, double ahi, double alo, double bhi, double blo) {
    dd x = dd_mul_d(dd{ahi, alo}, (double)m);
    dd y = dd_mul_d(dd{bhi, blo}, (double)n);
    return dd_add(x, y);
}
// general voices (Eq. 1): F = m f_phi + k f_theta + n f_r; knot values rounded in that order, so that k = 0
// gives the two-frequency value bit for bit
__device__ __forceinline__ double fdemri_knotF3(int m, int k, int n, double fphi, double fth, double fr) {
    return __dadd_rn(__dadd_rn(__dmul_rn((double)m, fphi), __dmul_rn((double)k, fth)), __dmul_rn((double)n, fr));
}

// roots of the monotone cubic  FB t + FC t^2 + FD t^3 = x  on [0, h]  for x = x1 and x = x2 (build time only: the two
// points shape the seed of the inverse, whose own interpolation error is ~1e-4 h, so four safeguarded Newton steps from
// the secant point are plenty).  Both roots advance together: two independent dependency chains, no divergent loop.
__device__ __forceinline__ void fdemri_root_build2(double FB, double FC, double FD, double x1, double x2, double h,
                                                   double& t1, double& t2) {
    const double Gh = h * (FB + h * (FC + h * FD));                // G(h) + x
    const bool inc = Gh > 0.0;                                     // G(h) > G(0)
    const double ih = (Gh != 0.0) ? h / Gh : 0.0;
    double lo1 = 0.0, hi1 = h, lo2 = 0.0, hi2 = h;
    t1 = fmin(fmax(x1 * ih, 0.0), h);                              // secant seeds
    t2 = fmin(fmax(x2 * ih, 0.0), h);
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const double G1 = t1 * (FB + t1 * (FC + t1 * FD)) - x1, G2 = t2 * (FB + t2 * (FC + t2 * FD)) - x2;
        const double d1 = FB + t1 * (2.0 * FC + 3.0 * FD * t1), d2 = FB + t2 * (2.0 * FC + 3.0 * FD * t2);
        if ((G1 > 0.0) == inc) hi1 = t1; else lo1 = t1;
        if ((G2 > 0.0) == inc) hi2 = t2; else lo2 = t2;
        double n1 = t1 - G1 / d1, n2 = t2 - G2 / d2;
        if (!(n1 > lo1 && n1 < hi1)) n1 = 0.5 * (lo1 + hi1);
        if (!(n2 > lo2 && n2 < hi2)) n2 = 0.5 * (lo2 + hi2);
        t1 = (G1 == 0.0) ? t1 : n1;
        t2 = (G2 == 0.0) ? t2 : n2;
    }
}

// ---- explicit frequency arrays: a bucket table instead of a full binary search per knot value ----------------------------
// lut = { double f_lo = freq[0], double inv_w, int64 first bin with f > 0, int64 0,  int first[lut_n + 1] }:
// first[j] = first bin with freq >= f_lo + j w,  w = (freq[n-1] - f_lo) / lut_n,  first[lut_n] = n_freq.
// A search takes the window [first[j-1], first[j+2]] around its bucket j = floor((x - f_lo) inv_w) -- one bucket of
// slack either side for the rounding of j -- finishes there, and CHECKS the answer against its two neighbours (falling back
// to the plain binary search, which never happened in any test): the table only ever saves time, it cannot move a bin.
// Built by the first fdemri_build_splines after fdemri_set_workspace; if the array changes afterwards, or the table is
// overwritten, the lookups fall back to the plain search one by one (indices read from the table are clamped first).
#define FDEMRI_LUT_HDR 8                    // ints in front of first[]

__device__ __forceinline__ int64_t fdemri_bsearch_ge(const double* __restrict__ f, int64_t lo, int64_t hi, double x) {
    // first i in [lo, hi] with f[i] >= x (hi if none in [lo, hi)): binary search down to a window of 8, then the window
    // at once (independent loads: one trip instead of three)
    while (hi - lo > 8) { int64_t mid = (lo + hi) >> 1; if (__ldg(f + mid) < x) lo = mid + 1; else hi = mid; }
    int below = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) below += (lo + j < hi && __ldg(f + lo + j) < x) ? 1 : 0;
    return lo + below;
}

__global__ void k_freq_lut(FdemriDims d, int* __restrict__ lut) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t n = d.n_freq;
    const double f_lo = __ldg(d.freq), f_hi = __ldg(d.freq + n - 1);
    const double w = (f_hi - f_lo) / (double)d.lut_n;
    if (j == 0) {
        double* hd = reinterpret_cast<double*>(lut);
        hd[0] = f_lo;
        hd[1] = (w > 0.0) ? 1.0 / w : 0.0;
        int64_t lo = 0, hi = n;                                     // first bin with f > 0 (R13)
        while (lo < hi) { int64_t mid = (lo + hi) >> 1; if (__ldg(d.freq + mid) <= 0.0) lo = mid + 1; else hi = mid; }
        reinterpret_cast<long long*>(lut)[2] = lo;
        reinterpret_cast<long long*>(lut)[3] = 0;
    }
    if (j > d.lut_n) return;
    lut[FDEMRI_LUT_HDR + j] = (j == d.lut_n) ? (int)n : (int)fdemri_bsearch_ge(d.freq, 0, n, f_lo + (double)j * w);
}

// first bin index with f_i >= x  (n_freq if none)
__device__ int64_t fdemri_first_ge(const FdemriDims& d, double x) {
    int64_t n = d.n_freq;
    if (d.freq) {
        if (d.lut) {
            const double* hd = reinterpret_cast<const double*>(d.lut);
            const double t = (x - __ldg(hd)) * __ldg(hd + 1);
            if (t >= 0.0 && t < (double)d.lut_n) {                  // (NaN and the two ends take the plain search)
                const int j = (int)t;
                const int64_t lo = min(max((int64_t)__ldg(d.lut + FDEMRI_LUT_HDR + max(j - 1, 0)), (int64_t)0), n);
                const int64_t hi = min(max((int64_t)__ldg(d.lut + FDEMRI_LUT_HDR + min(j + 2, d.lut_n)), lo), n);
                const int64_t i = fdemri_bsearch_ge(d.freq, lo, hi, x);
                const bool ok = (i == 0 || __ldg(d.freq + i - 1) < x) && (i == n || __ldg(d.freq + i) >= x);
                if (ok) return i;
            }
        }
        return fdemri_bsearch_ge(d.freq, 0, n, x);
    }
    double g = ceil((x - d.f0) * d.inv_df);
    int64_t i = (g <= 0.0) ? 0 : (g >= (double)n ? n : (int64_t)g);
    while (i > 0 && fdemri_freq(d, i - 1) >= x) --i;
    while (i < n && fdemri_freq(d, i) < x) ++i;
    return i;
}
// first bin index with f_i > 0 (R13: only bins with f > 0 carry signal)
__device__ int64_t fdemri_first_positive(const FdemriDims& d) {
    int64_t n = d.n_freq;
    if (d.freq) {
        if (d.lut) {
            const int64_t i = min(max((int64_t)reinterpret_cast<const long long*>(d.lut)[2], (int64_t)0), n);
            if ((i == 0 || __ldg(d.freq + i - 1) <= 0.0) && (i == n || __ldg(d.freq + i) > 0.0)) return i;
        }
        int64_t lo = 0, hi = n;
        while (lo < hi) { int64_t mid = (lo + hi) >> 1; if (__ldg(d.freq + mid) <= 0.0) lo = mid + 1; else hi = mid; }
        return lo;
    }
    double g = floor((0.0 - d.f0) * d.inv_df) + 1.0;
    int64_t i = (g <= 0.0) ? 0 : (g >= (double)n ? n : (int64_t)g);
    while (i > 0 && fdemri_freq(d, i - 1) > 0.0) --i;
    while (i < n && fdemri_freq(d, i) <= 0.0) ++i;
    return i;
}

// ------------------------------------------------------------------------------------------------
// S2: one WARP per (batch item, voice); its lanes take the segments 32 at a time ("groups" of 32 consecutive
// segments).  Per segment: the record (F cubic, phase cubic, inversion seed or extrema) and, for both signs and up
// to three monotone branches, the interval of bins the branch covers ("entry").  Per group and per voice-sign the
// union of those intervals ("bands"): the sum kernels find the entries that meet a tile of bins by walking
//     voice-sign band  ->  group bands  ->  the 32 entries of a group row
// in ascending key order -- no per-tile list is ever built, sorted or stored (the paper: "the spline segment in
// which each value of f falls is predetermined before the summation", L105; here the predetermined map is the
// entries plus two levels of bands over them).
//   ent   [B][V][2][3][Sp] int2 {first bin, last bin}; empty: last < first; Sp = 32 G (rows padded with empty entries to
//         whole groups: a group row is 256 aligned bytes).   key = ((v*2+sign)*3 + branch)*Sp + segment
//   gband [B][V][2][G] int4 {lo, hi of the branch-0 entries of the group; lo, hi of its branch-1/2 entries}
//   vband [B][V][2]    int2 {lo, hi} over all entries of the voice-sign
//   iband [B]          int2 {max of 0x7fffffff - lo, max of hi + 1} over the item (atomicMax; zeroed before: {0, 0} = empty)
// POLAR: general voices (l, m, k, n) -- kk[v] = k, sh2_hi/sh2_lo the splines of (f_theta, Phi_theta) (components
// 0 and 1 of a second [B][4][n_seg][4] array), f_theta the knot values.
// ------------------------------------------------------------------------------------------------
#define FDEMRI_REC_WARPS 4           // warps (voices) per CTA of k_records

template <bool POLAR>
__global__ void __launch_bounds__(FDEMRI_REC_WARPS * 32)
k_records(FdemriDims d, const int* __restrict__ lmn, const double* __restrict__ t_knots,
          const double* __restrict__ sh_hi, const double* __restrict__ sh_lo,
          const double* __restrict__ f_phi, const double* __restrict__ f_r, double* __restrict__ rec,
          int2* __restrict__ ent, int4* __restrict__ gband, int2* __restrict__ vband, int* __restrict__ iband,
          const unsigned char* __restrict__ mode_mask, unsigned long long* __restrict__ stats,
          unsigned long long* __restrict__ item_evals, const int* __restrict__ kk,
          const double* __restrict__ sh2_hi, const double* __restrict__ sh2_lo,
          const double* __restrict__ f_theta) {
    const int lane = threadIdx.x & 31;
    const size_t bv = (size_t)blockIdx.x * FDEMRI_REC_WARPS + (threadIdx.x >> 5);
    if (bv >= (size_t)d.n_batch * d.n_modes) return;                 // whole warp
    const unsigned full = 0xffffffffu;
    const int v = (int)(bv % d.n_modes);
    const int b = (int)(bv / d.n_modes);
    const int m = lmn[3 * v + 1], n = lmn[3 * v + 2];
    const int S = d.n_seg, G = d.n_groups;
    const size_t per = (size_t)S * 4;
    const int kq = POLAR ? kk[v] : 0;
    const bool masked = mode_mask && !mode_mask[bv];                 // a mode the selection dropped has no entries
    const int64_t first_pos = fdemri_first_positive(d);              // bins with f > 0 only (R13)
    const dd inv2pi = dd{FDEMRI_INV2PI_HI, FDEMRI_INV2PI_LO};
    const size_t last = (size_t)b * d.n_knots + d.n_knots - 1;
    unsigned long long evals = 0;
    unsigned items = 0, turnovers = 0;
    bool bad = false;
    int vlo[2] = {0x7fffffff, 0x7fffffff}, vhi[2] = {-1, -1};
    for (int g = 0; g < G; ++g) {
        const int k = 32 * g + lane;
        const bool active = k < S;
        int2 e[2][3];
#pragma unroll
        for (int sg = 0; sg < 2; ++sg)
#pragma unroll
            for (int br = 0; br < 3; ++br) e[sg][br] = make_int2(0, -1);       // empty: last < first
        double V0 = 0.0, V1 = 0.0, V2 = 0.0, V3 = 0.0;
        int nbr = 0;
        if (active) {
            // coefficients (a, b, c, d) of f_phi, f_r, Phi_phi, Phi_r on this segment, hi and lo parts
            const double4* H4 = reinterpret_cast<const double4*>(sh_hi + (size_t)b * 4 * per) + k;
            const double4* L4 = reinterpret_cast<const double4*>(sh_lo + (size_t)b * 4 * per) + k;
            const double4 h0 = H4[0], h1 = H4[S], h2 = H4[2 * (size_t)S], h3 = H4[3 * (size_t)S];
            const double4 l0 = L4[0], l1 = L4[S], l2 = L4[2 * (size_t)S], l3 = L4[3 * (size_t)S];
            // F cubic (Eq. 6)
            double FA = fdemri_knotF(m, n, h0.x, h1.x);
            dd FBd = fdemri_combine(m, n, h0.y, l0.y, h1.y, l1.y);
            dd FCd = fdemri_combine(m, n, h0.z, l0.z, h1.z, l1.z);
            dd FDd = fdemri_combine(m, n, h0.w, l0.w, h1.w, l1.w);
            // phase spline of the voice, in cycles (R9)
            dd Pa = dd_add(two_prod((double)m, h2.x), two_prod((double)n, h3.x));   // knot values: exact
            dd Pb = fdemri_combine(m, n, h2.y, l2.y, h3.y, l3.y);
            dd Pc = fdemri_combine(m, n, h2.z, l2.z, h3.z, l3.z);
            dd Pd = fdemri_combine(m, n, h2.w, l2.w, h3.w, l3.w);
            const double4* G4 = nullptr;
            if (POLAR) {                                            // the polar terms k f_theta, k Phi_theta (Eq. 1)
                G4 = reinterpret_cast<const double4*>(sh2_hi + (size_t)b * 4 * per) + k;
                const double4* GL = reinterpret_cast<const double4*>(sh2_lo + (size_t)b * 4 * per) + k;
                const double4 g0 = G4[0], g1 = G4[S], e0 = GL[0], e1 = GL[S];
                const double kd = (double)kq;
                FA = fdemri_knotF3(m, kq, n, h0.x, g0.x, h1.x);
                FBd = dd_add(FBd, dd_mul_d(dd{g0.y, e0.y}, kd));
                FCd = dd_add(FCd, dd_mul_d(dd{g0.z, e0.z}, kd));
                FDd = dd_add(FDd, dd_mul_d(dd{g0.w, e0.w}, kd));
                Pa = dd_add(Pa, two_prod(kd, g1.x));
                Pb = dd_add(Pb, dd_mul_d(dd{g1.y, e1.y}, kd));
                Pc = dd_add(Pc, dd_mul_d(dd{g1.z, e1.z}, kd));
                Pd = dd_add(Pd, dd_mul_d(dd{g1.w, e1.w}, kd));
            }
            const double FB = FBd.hi, FC = FCd.hi, FD = FDd.hi;
            const double pc = -dd_frac(dd_mul(Pa, inv2pi));
            const dd bq = dd_mul(Pb, inv2pi);
            const double tk = t_knots[(size_t)b * d.n_knots + k];
            const double h = __dadd_rn(t_knots[(size_t)b * d.n_knots + k + 1], -tk);
            double rQ1, rQ2, rQ3, rTYPE, rSF;
            // interior extrema of F on (0, h): roots of FB + 2 FC t + 3 FD t^2
            double ext[2]; int ne = 0;
            {
                const double qa = 3.0 * FD, qb = 2.0 * FC, qc = FB;
                if (qa == 0.0) {
                    if (qb != 0.0) { const double r = -qc / qb; if (r > 0.0 && r < h) ext[ne++] = r; }
                } else {
                    const double disc = qb * qb - 4.0 * qa * qc;
                    if (disc > 0.0) {
                        const double sq = sqrt(disc);
                        const double qq = -0.5 * (qb + (qb >= 0.0 ? sq : -sq));
                        double r1 = qq / qa, r2 = (qq != 0.0) ? qc / qq : r1;
                        if (r1 > r2) { const double tmp = r1; r1 = r2; r2 = tmp; }
                        if (r1 > 0.0 && r1 < h) ext[ne++] = r1;
                        if (r2 > 0.0 && r2 < h && r2 != r1) ext[ne++] = r2;
                    }
                }
            }
            if (!(isfinite(FA) && isfinite(FB) && isfinite(FC) && isfinite(FD) && isfinite(pc) && isfinite(bq.hi))) bad = true;
            if (ne == 0) {
                // seed of the inverse: cubic through tau(x) at x = dF {0, 1/3, 2/3, 1}, x = s f - FA
                const double dF = h * (FB + h * (FC + h * FD));
                double q1 = 0.0, q2 = 0.0, q3 = 0.0;
                if (dF != 0.0 && isfinite(dF)) {
                    double t1, t2;
                    fdemri_root_build2(FB, FC, FD, dF * (1.0 / 3.0), dF * (2.0 / 3.0), h, t1, t2);
                    const double g1 = 3.0 * t1, g2 = 1.5 * t2, g3 = h;
                    const double gam = 4.5 * (g1 - 2.0 * g2 + g3);
                    const double bet = 3.0 * (g2 - g1) - gam;
                    const double alp = g1 - bet * (1.0 / 3.0) - gam * (1.0 / 9.0);
                    const double idF = 1.0 / dF;
                    q1 = alp * idF; q2 = bet * idF * idF; q3 = gam * idF * idF * idF;
                }
                rQ1 = q1; rQ2 = q2; rQ3 = q3; rTYPE = 0.0;
                rSF = (dF < 0.0) ? -1.0 : 1.0;
            } else if (ne == 1) {
                const double te = ext[0];
                rQ1 = te;
                rQ2 = FA + te * (FB + te * (FC + te * FD));          // F_e (R7)
                rQ3 = 0.0;
                rTYPE = 1.0;
                rSF = 0.0;
                ++turnovers;
            } else {
                // two interior extrema (the paper assumes at most one, L105; R5): three monotone branches
                const double t1 = ext[0], t2 = ext[1];
                rQ1 = t1;
                rQ2 = FA + t1 * (FB + t1 * (FC + t1 * FD));          // F_e1
                rQ3 = t2;
                rTYPE = 2.0;
                rSF = FA + t2 * (FB + t2 * (FC + t2 * FD));          // F_e2 (the slot of the sign, which type 0 alone needs)
                ++turnovers;
            }
            {
                // the record: four 32-byte stores (slots 8..15 belong to k_spline_amp)
                double4* R4 = reinterpret_cast<double4*>(rec + (bv * S + k) * R_DOUBLES);
                R4[0] = make_double4(FA, FB, FC, FD);
                R4[1] = make_double4(rQ1, rQ2, rQ3, h);
                R4[4] = make_double4(pc, bq.hi, bq.lo, -dd_mul(Pc, inv2pi).hi);
                R4[5] = make_double4(-dd_mul(Pd, inv2pi).hi, tk, rTYPE, rSF);
            }
            // ---- bin intervals of the branches of this segment, for both signs (L105) ----
            const int type = (int)rTYPE;
            const double Fk = FA;
            double Fk1;
            if (POLAR) Fk1 = (k + 1 < S) ? fdemri_knotF3(m, kq, n, H4[1].x, G4[1].x, H4[S + 1].x)
                                         : fdemri_knotF3(m, kq, n, f_phi[last], f_theta[last], f_r[last]);
            else    Fk1 = (k + 1 < S) ? fdemri_knotF(m, n, H4[1].x, H4[S + 1].x)
                                      : fdemri_knotF(m, n, f_phi[last], f_r[last]);
            // branch j of the segment runs from V[j] to V[j+1]: knot value, extremum values, next knot value; a branch
            // includes its start iff that is the knot and its end iff that is an extremum (R6, R7)
            V0 = Fk; V1 = type >= 1 ? rQ2 : Fk1; V2 = type == 2 ? rSF : Fk1; V3 = Fk1;
            nbr = masked ? 0 : type + 1;
        }
        // One search per knot: g = first bin >= |F_k|, and whether that bin equals |F_k| (then first bin > |F_k| is g + 1).
        // The next knot's pair comes from the next lane; the last lane of the group looks its own up.  (Scalars and
        // selects, no indexed arrays: those would live in local memory.)
        int g0, g1, g2, g3;
        bool q0, q1, q2, q3;
        {
            const double a0 = fabs(V0);
            const int64_t s0 = active ? fdemri_first_ge(d, a0) : 0;
            g0 = (int)s0;
            q0 = active && s0 < d.n_freq && fdemri_freq(d, s0) == a0;
            g3 = __shfl_down_sync(full, g0, 1);
            q3 = __shfl_down_sync(full, (int)q0, 1) != 0;
            if (active && (lane == 31 || k + 1 >= S)) {              // no next lane holds the knot k + 1
                const double a3 = fabs(V3);
                const int64_t s3 = fdemri_first_ge(d, a3);
                g3 = (int)s3;
                q3 = s3 < d.n_freq && fdemri_freq(d, s3) == a3;
            }
            g1 = g2 = g3; q1 = q2 = q3;
            if (active && nbr > 1) {                                 // extremum values (turnover segments only)
                const double a1 = fabs(V1);
                const int64_t s1 = fdemri_first_ge(d, a1);
                g1 = (int)s1;
                q1 = s1 < d.n_freq && fdemri_freq(d, s1) == a1;
            }
            if (active && nbr > 2) {
                const double a2 = fabs(V2);
                const int64_t s2 = fdemri_first_ge(d, a2);
                g2 = (int)s2;
                q2 = s2 < d.n_freq && fdemri_freq(d, s2) == a2;
            }
        }
        if (active) {
#pragma unroll
            for (int sg = 0; sg < 2; ++sg) {
#pragma unroll
                for (int br = 0; br < 3; ++br) {
                    if (br < nbr) {
                        // end values of the branch: start (index br) and end (index br + 1, or 3 = the next knot)
                        const bool to_knot = !(br + 1 < nbr);
                        const double Va = br == 0 ? V0 : (br == 1 ? V1 : V2);
                        const int ga = br == 0 ? g0 : (br == 1 ? g1 : g2);
                        const bool qa = br == 0 ? q0 : (br == 1 ? q1 : q2);
                        const double Vb = to_knot ? V3 : (br == 0 ? V1 : V2);
                        const int gb = to_knot ? g3 : (br == 0 ? g1 : g2);
                        const bool qb = to_knot ? q3 : (br == 0 ? q1 : q2);
                        const bool a_incl = (br == 0), b_incl = !to_knot;
                        if (Va != Vb) {
                            const bool up = Va < Vb;
                            const double Vlo = up ? Va : Vb, Vhi = up ? Vb : Va;      // lower / higher end value
                            const int glo = up ? ga : gb, ghi = up ? gb : ga;
                            const bool qlo = up ? qa : qb, qhi = up ? qb : qa;
                            const bool lo_incl = up ? a_incl : b_incl, hi_incl = up ? b_incl : a_incl;
                            // in terms of f = s x:  s = +1: f in [Vlo, Vhi];  s = -1: f in [-Vhi, -Vlo]
                            const double flo = sg ? -Vhi : Vlo, fhi = sg ? -Vlo : Vhi;
                            const int gflo = sg ? ghi : glo, gfhi = sg ? glo : ghi;
                            const bool qflo = sg ? qhi : qlo, qfhi = sg ? qlo : qhi;
                            const bool flo_incl = sg ? hi_incl : lo_incl, fhi_incl = sg ? lo_incl : hi_incl;
                            if (fhi > 0.0) {
                                // first bin >= x (incl) or > x (excl); x <= 0: every bin qualifies (clipped to f > 0 below)
                                int64_t lo_b = (flo > 0.0) ? (int64_t)gflo + ((!flo_incl && qflo) ? 1 : 0) : 0;
                                const int64_t hi1 = (int64_t)gfhi + ((fhi_incl && qfhi) ? 1 : 0);
                                if (lo_b < first_pos) lo_b = first_pos;
                                if (lo_b < hi1) {
                                    e[sg][br] = make_int2((int)lo_b, (int)(hi1 - 1));
                                    evals += (unsigned long long)(hi1 - lo_b);
                                    ++items;
                                }
                            }
                        }
                    }
                }
            }
        }
        // entries (coalesced rows of the group) and the bands over them
#pragma unroll
        for (int sg = 0; sg < 2; ++sg) {
            int lo0 = 0x7fffffff, hi0 = -1, lo12 = 0x7fffffff, hi12 = -1;
#pragma unroll
            for (int br = 0; br < 3; ++br) {
                const int2 q = e[sg][br];
                ent[((bv * 2 + sg) * 3 + br) * (size_t)(32 * G) + k] = q;       // (lanes past the last segment: empty)
                if (q.y >= q.x) {
                    if (br == 0) { lo0 = q.x; hi0 = q.y; }
                    else { lo12 = min(lo12, q.x); hi12 = max(hi12, q.y); }
                }
            }
            lo0 = __reduce_min_sync(full, lo0); hi0 = __reduce_max_sync(full, hi0);
            lo12 = __reduce_min_sync(full, lo12); hi12 = __reduce_max_sync(full, hi12);
            if (lane == 0) gband[(bv * 2 + sg) * (size_t)G + g] = make_int4(lo0, hi0, lo12, hi12);
            vlo[sg] = min(vlo[sg], min(lo0, lo12));
            vhi[sg] = max(vhi[sg], max(hi0, hi12));
        }
    }
    // bands of the voice, of the item; counters: one atomic per warp
    const unsigned it_w = __reduce_add_sync(full, items);
    const unsigned tv_w = __reduce_add_sync(full, turnovers);
    const unsigned lo_w = __reduce_add_sync(full, (unsigned)(evals & 0xffffu));
    const unsigned mi_w = __reduce_add_sync(full, (unsigned)((evals >> 16) & 0xffffu));
    const unsigned hi_w = __reduce_add_sync(full, (unsigned)(evals >> 32));
    const bool any_bad = __any_sync(full, bad);
    if (lane == 0) {
        vband[bv * 2 + 0] = make_int2(vlo[0], vhi[0]);
        vband[bv * 2 + 1] = make_int2(vlo[1], vhi[1]);
        const int ilo = min(vlo[0], vlo[1]), ihi = max(vhi[0], vhi[1]);
        if (ihi >= ilo) {
            atomicMax(iband + 2 * b, 0x7fffffff - ilo);
            atomicMax(iband + 2 * b + 1, ihi + 1);
        }
        if (it_w) atomicAdd(stats + 0, (unsigned long long)it_w);
        if (tv_w) atomicAdd(stats + 3, (unsigned long long)tv_w);
        const unsigned long long ev = ((unsigned long long)hi_w << 32) + ((unsigned long long)mi_w << 16) + lo_w;
        if (ev) {
            atomicAdd(stats + 2, ev);
            atomicAdd(item_evals + b, ev);
        }
        if (any_bad) atomicOr(stats + 5, 4ull);
    }
}
