// fdemri_sum.cuh -- S3 + S4: the output-tiled harmonic sum (the hot loop).
//
// A CTA owns a tile of FDEMRI_TILE consecutive bins of one batch item at a time (tiles are handed out by an
// atomic counter).  It is warp-specialised:
//   * one PRODUCER warp finds the entries -- (voice, sign, segment-branch) -- that intersect the tile by walking the
//     bands of fdemri_map.cuh (voice-sign band -> group bands -> the 32 entries of a group row) in ascending key
//     order, reads their records and weights from global memory, folds everything that does not depend on the bin
//     into a 256-byte staged item, and pushes chunks of staged items through a shared-memory ring (full/empty
//     mbarriers).  No per-tile list exists anywhere: the walk is the list;
//   * FDEMRI_CWARPS CONSUMER warps each own 64 consecutive bins of the tile, two per lane (lane, lane + 32),
//     with the eight accumulators in registers.  For every staged item that overlaps its bins a consumer warp
//     evaluates the term of Eq. 9 for both of its bins at once (two independent
//     dependency chains per thread hide the 8-cycle FP64 latency):
//         A(t) g(X)/sqrt|Fdot| exp{i[2 pi s f t - Phi(t)]},   t = t_k + tau,  F(tau) = s f  (Eq. 6)
//     and adds it with the harmonic weights (Eq. 1).
// Every bin is written once (S4): no atomics on the data path, and the summation order of a bin depends only
// on the data, never on scheduling: results are bitwise reproducible.
// The paper's own layout -- one block per (voice, segment), atomicAdd into global memory (L121) -- is prior art.
//
// Fast path (monotone segment, |X| >= 400, ~99 % of the evaluations): division-free inversion of the segment
// cubic -- stored inverse-cubic seed and one Halley step in SINGLE precision (FMA pipe), then one FP64 Newton
// correction whose size is the acceptance test -- then the polar form of the asymptotic g(X) series and a
// polynomial sincos of the phase in quarter turns.  The FP64 pipe is the bound (a DFMA with three distinct
// register operands issues every 3 cycles, not 2: see profiles/), so everything that tolerates it runs elsewhere.
// Everything else (turnover segments, small |X|, rejected iterations) goes to fdemri_term_slow.
#pragma once
#include "fdemri_common.cuh"
#include "airy_tables.inc"
#include "poly_tables.inc"

#ifndef FDEMRI_CONS_BACKOFF
#define FDEMRI_CONS_BACKOFF 64u     // ns between polls of a consumer warp waiting for a stage
#endif
#ifndef FDEMRI_PROD_BACKOFF
#define FDEMRI_PROD_BACKOFF 1000u   // ns between polls of the producer warp waiting for a free stage (it runs stages ahead)
#endif

struct SumArgs {
    FdemriDims d;
    const double* rec;        // [B][V][S][R_DOUBLES]
    const int2* ent;          // [B][V][2][3][Sp] {first bin, last bin}, Sp = 32 G; key = ((v*2+sign)*3 + branch)*Sp + segment
    const int4* gband;        // [B][V][2][G] bands of the groups of 32 segments {lo, hi (branch 0), lo, hi (branches 1, 2)}
    const int2* vband;        // [B][V][2] band of the voice-sign
    const int* iband;         // [B][2] {0x7fffffff - lo, hi + 1} of the item ({0, 0}: empty)
    const double4* wts;       // [n_angles][V]
    int n_angles;
    double* hp;               // [B][n_freq][2]
    double* hx;
    unsigned int* tile_counter;
    unsigned long long* stats;
    int total_tiles;
    // fused inner products (Eq. 12): all NULL for a plain sum
    const double* weight;     // [n_freq] w_k = 4 df / S_n(f_k), or NULL for w = 1
    const double* dplus;      // [n_freq][2] data, + polarisation (NULL: only <h|h>)
    const double* dcross;     // [n_freq][2]
    double* inner_part;       // [ranges][4] partial sums {<h|h>, Re<d|h>, Im<d|h>, 0}; a range = the 64 bins of a consumer
                              // warp (tile-major: total_tiles * FDEMRI_CWARPS ranges) or a block of bins (bin-major)
    double* inner_edge;       // Hann filter (L145): [ranges][4][4] h at the first two and last two bins of every range;
                              // NULL: no window
};

// asymptotic series of g(X) e^{+i pi/4 sgn X} = sum_k i^k a_k u^k, u = 1/X, a_k = prod_j (4/9-(2j-1)^2)/(k! 8^k)
__constant__ double c_gre[7] = {1.0, -0.037133487654320986, 0.05764919041266972, -0.2915913992307505,
                                3.079453030173167, -55.62278536591708, 1533.1694320127956};
__constant__ double c_gim[6] = {-0.06944444444444445, 0.03799305912780064, -0.11609906402551541,
                                0.8776669695100169, -12.341573332345238, 278.46508077760257};

// x with its sign bit XORed by `mask` (0 or 0x80000000): one integer op on the high word
__device__ __forceinline__ double fdemri_xorsign(double x, unsigned mask) {
    return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}

// high word of |x|: monotone in |x| for finite x, and larger than any finite threshold for NaN/Inf
__device__ __forceinline__ int fdemri_hiabs(double x) { return __double2hiint(x) & 0x7fffffff; }

// sin, cos of q quarter turns (|q| up to ~1e4; absolute error ~1e-14 + (pi/2) ulp(q))
__device__ __forceinline__ void fdemri_sincos_quarter(double q, double& sn, double& cs) {
    const double big = 6755399441055744.0;             // 1.5 * 2^52: adding it rounds to the nearest integer
    const double t = q + big;
    const int k = __double2loint(t);                   // low word of the sum = the integer (two's complement)
    const double r = q - (t - big);                    // in [-1/2, 1/2], exact
    const double r2 = r * r;
    double s = c_sinq[FDEMRI_NSIN - 1];
#pragma unroll
    for (int i = FDEMRI_NSIN - 2; i >= 0; --i) s = fma(s, r2, c_sinq[i]);
    s *= r;
    double co = c_cosq[FDEMRI_NCOS - 1];
#pragma unroll
    for (int i = FDEMRI_NCOS - 2; i >= 0; --i) co = fma(co, r2, c_cosq[i]);
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

// ~21 good bits of |a|^(-1/2) (MUFU.RSQ64H reads the high word only; the sign is cleared with an integer op)
__device__ __forceinline__ double fdemri_rsqrt_seed_abs(double a) {
    double y;
    const double aa = __hiloint2double(__double2hiint(a) & 0x7fffffff, 0);
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(aa));
    return y;
}

// ---- mbarrier helpers (shared::cta) ----------------------------------------------------------------------
__device__ __forceinline__ unsigned fdemri_smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fdemri_mbar_init(uint64_t* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(fdemri_smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fdemri_mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(fdemri_smem_addr(bar)) : "memory");
}
__device__ __forceinline__ bool fdemri_mbar_try(unsigned addr, unsigned parity) {
    unsigned done;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(addr), "r"(parity)
        : "memory");
    return done != 0u;
}
// spin with a back-off of `ns` nanoseconds between polls (a polling warp takes issue slots from its SM sub-partition)
__device__ __forceinline__ void fdemri_mbar_wait(uint64_t* bar, unsigned parity, unsigned ns) {
    const unsigned addr = fdemri_smem_addr(bar);
    while (!fdemri_mbar_try(addr, parity)) __nanosleep(ns);
}

// ---------------------------------------------------------------------------------------------------------
// Fast path of one term.  it: the staged item (shared memory); sf = s f.  Returns T = A g/sqrt|F'| e^{i psi}
// and ok = the inversion was accepted and |X| >= 400.  Branch-free, so two calls interleave.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool fdemri_term_fast(const double* __restrict__ it, double sf, double& Tre, double& Tim) {
    const double FB = it[S_FB], FC = it[S_FC], FD = it[S_FD];
    const double x = sf + it[S_NFA];
    // First iterate in SINGLE precision (FMA pipe, not the FP64 pipe): stored inverse-cubic seed, then a Halley
    // step  tau <- tau - d (1 + d F''/(2 F')),  d = G/F'.  It only has to land within ~1e-7 h of the root.
    double tau;
    {
        const float2 c0 = *reinterpret_cast<const float2*>(it + S_F32A);      // FB, FC
        const float2 c1 = *reinterpret_cast<const float2*>(it + S_F32B);      // FD, Q1
        const float2 c2f = *reinterpret_cast<const float2*>(it + S_F32C);     // Q2, Q3
        const float xf = (float)x;
        float tf = xf * fmaf(xf, fmaf(xf, c2f.y, c2f.x), c1.y);
        const float b2 = fmaf(tf, c1.x, c0.y), b1 = fmaf(tf, b2, c0.x), G = fmaf(tf, b1, -xf);
        const float c2 = fmaf(tf, c1.x, b2), dG = fmaf(tf, c2, b1), Fh = fmaf(tf, c1.x, c2);
        float r;
        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(dG));
        const float d0 = G * r;
        tf = fmaf(-d0, d0 * (Fh * r), tf - d0);
        tau = (double)tf;
    }
    // Newton correction at the new point; its size is the acceptance test
    const double b2 = fma(tau, FD, FC), b1 = fma(tau, b2, FB), G = fma(tau, b1, -x);
    const double c2 = fma(tau, FD, b2), dG = fma(tau, c2, b1), Fh = fma(tau, FD, c2);   // Fh = F''/2
    double y = fdemri_rsqrt_seed_abs(dG);
    {   // second-order refinement of y ~ |F'|^(-1/2): y (1 + e/2), e = 1 - |F'| y^2; relative error 2^-22 -> 3/8 e^2 < 1e-13
        const double t = fabs(dG) * y;
        const double he = fma(-t, 0.5 * y, 0.5);
        y = fma(y, he, y);
    }
    const double r = y * y;                            // 1/|F'|
    const double rs = copysign(r, dG);
    const double delta = G * rs;
    tau -= delta;
    // values at the corrected point, to first order in delta (second order is below 1e-13):
    //   F''/2 -> Fh - 3 FD delta,   F' -> F' (1 - 2 tq),  tq = delta (Fh - 1.5 FD delta) / F',   |F'|^(-1/2) -> y (1 + tq)
    const double t3 = delta * FD;
    const double Fhc = fma(t3, -3.0, Fh);
    const double tq = (delta * fma(t3, -1.5, Fh)) * rs;
    y = fma(y, tq, y);
    // accept: the neglected second-order terms are below rounding (|F'' delta / F'| <= 5e-7 and |delta| <= 2e-7 h)
    // and the iterate sits in the segment (the root does, by membership R6)
    // (compared on the high words: |v| <= T  <=>  hi(|v|) <= hi(T) up to 2^-20 relative; NaN fails)
    const double rc = y * y;                           // 1/|F'| at the corrected point
    const double pq = Fhc * rc;
    const double u = (pq * pq) * (rc * it[S_CU]);      // 1/X = 3 F''^2 / (2 pi F'^3), needed to 1e-9 relative
    const bool ok = (fdemri_hiabs(tq) <= 0x3e90c6f7) & (fdemri_hiabs(delta) <= __double2hiint(it[S_TOLH])) &
                    (fdemri_hiabs(tau - it[S_HH]) <= __double2hiint(it[S_HH])) & (fdemri_hiabs(u) <= 0x3f647ae1);
    const double u2 = u * u;
    const double dq = u * fma(u2, FDEMRI_G_DQ3, FDEMRI_G_DQ1);
    const double yr = y * fma(u2, FDEMRI_G_R2, 1.0);        // (the u^4 term of rho is below 2.2e-12 for |X| >= 400)
    // amplitude (two cubics)
    const double Are = fma(tau, fma(tau, fma(tau, it[S_AR + 3], it[S_AR + 2]), it[S_AR + 1]), it[S_AR]);
    const double Aim = fma(tau, fma(tau, fma(tau, it[S_AI + 3], it[S_AI + 2]), it[S_AI + 1]), it[S_AI]);
    // phase in quarter turns (R9): (s f)(4 t_k) exactly as P + e, P reduced modulo 4; local cubic in tau
    const double TK4 = it[S_TK4];
    const double P = __dmul_rn(sf, TK4);
    const double e = __fma_rn(sf, TK4, -P);
    const double big4 = 27021597764222976.0;           // 1.5 * 2^54: adding it rounds to a multiple of 4
    const double pr = P - ((P + big4) - big4);
    const double wv = fma(x, 4.0, it[S_WC]);           // 4 (s f - b'), b' = Phi'(t_k)/2pi, through x = s f - F_k
    const double loc = fma(tau, fma(tau, fma(tau, it[S_ND4], it[S_NC4]), wv), it[S_PC4]);
    const double q = (pr + e) + (loc + dq);
    double sn, cs;
    fdemri_sincos_quarter(q, sn, cs);
    const double Er = yr * cs, Ei = yr * sn;
    Tre = Are * Er - Aim * Ei;
    Tim = Are * Ei + Aim * Er;
    return ok;
}

// ---------------------------------------------------------------------------------------------------------
// Slow path of one term: turnover segments, small |X| (long series or Airy form), rejected fast iterations.
// flags: bit 0 branch of a segment with extrema, bit 1 it hangs between two extrema, bit 2 sign.  Returns T and
// counters in `info`:
// bit 0 Airy form used, bit 1 monotone fallback Newton, bits 4.. error bits (FDEMRI_BAD_NEWTON << 4).
// ---------------------------------------------------------------------------------------------------------
struct FdemriSlowOut {
    double tre, tim;
    unsigned info;
};

__device__ __noinline__ FdemriSlowOut fdemri_term_slow(const double* it, double sf, unsigned flags) {
    FdemriSlowOut out;
    out.tre = 0.0; out.tim = 0.0; out.info = 0u;
    const double FB = it[S_FB], FC = it[S_FC], FD = it[S_FD];
    const double h = 2.0 * it[S_HH];
    double tau, Fd, Fdd;
    if (!(flags & 1u)) {
        // monotone segment: safeguarded Newton with a true division from the stored seed
        const double x = sf + it[S_NFA];
        tau = x * fma(x, fma(x, it[S_Q3], it[S_Q2]), it[S_Q1]);
        tau = fmin(fmax(tau, 0.0), h);
        double dG = 0.0, c2 = 0.0;
        int n = 0;
        double prev = h;
        for (; n < 60; ++n) {
            const double b2 = fma(tau, FD, FC), b1 = fma(tau, b2, FB), G = fma(tau, b1, -x);
            c2 = fma(tau, FD, b2); dG = fma(tau, c2, b1);
            const double delta = G / dG;
            if (!(fabs(delta) > 1e-14 * h)) { if (fabs(delta) <= h) tau -= delta; break; }
            const double tn = fmin(fmax(tau - delta, 0.0), h);
            // no progress any more: the root sits on an end of the segment (the step is clamped away), or the step has
            // reached its rounding floor -- the iterate is as good as it gets
            if (tn == tau || (fabs(delta) >= prev && fabs(delta) <= 1e-9 * h)) { tau = tn; break; }
            prev = fabs(delta);
            tau = tn;
        }
        if (n == 60) out.info |= (8u << 4);
        tau = fmin(fmax(tau, 0.0), h);
        {
            const double b2 = fma(tau, FD, FC), b1 = fma(tau, b2, FB);
            c2 = fma(tau, FD, b2); Fd = fma(tau, c2, b1);
        }
        Fdd = 2.0 * fma(tau, FD, c2);
        out.info |= 2u;
    } else {
        // branch of a segment with extrema, bracket [ta, tb]: around the extremum it hangs on (the nearer one in value
        // when it hangs between two)  F(tau) - F_e = z^2 (c2 + FD z),  z = tau - tau_e
        const double ta = it[S_F32A], tb = it[S_F32B];
        double te = it[S_Q1], Fe = it[S_Q2], c2 = it[S_Q3];
        if ((flags & 2u) && fabs(sf - it[S_FREE]) < fabs(sf - Fe)) { te = it[S_F32C]; Fe = it[S_FREE]; c2 = it[S_TOLH]; }
        const double Delta = sf - Fe;
        double z = sqrt(fmax(Delta / c2, 0.0));
        if (0.5 * (ta + tb) < te) z = -z;
        const double tol = 1e-14 * h;
        int n = 0;
        double prev = h;
        for (; n < 40; ++n) {
            const double H = fma(z * z, fma(FD, z, c2), -Delta);
            const double dH = z * fma(3.0 * FD, z, 2.0 * c2);
            if (dH == 0.0) break;
            const double delta = H / dH;
            z -= delta;
            if (fabs(delta) <= tol) break;
            if (fabs(delta) >= prev && fabs(delta) <= 1e-9 * h) break;       // rounding floor of the step
            prev = fabs(delta);
        }
        if (n == 40) out.info |= (8u << 4);
        tau = fmin(fmax(te + z, ta), tb);
        z = tau - te;
        Fd = z * fma(3.0 * FD, z, 2.0 * c2);          // exact factorisation, no cancellation near Fdot = 0
        Fdd = fma(6.0 * FD, tau, 2.0 * FC);
    }
    if (Fd == 0.0 && Fdd == 0.0) return out;           // R10: no term
    const double aFd = fabs(Fd);
    const bool series = 6.283185307179586 * aFd * aFd * aFd >= 84.0 * Fdd * Fdd;      // |X| >= 28
    // amplitude
    const double Are = fma(tau, fma(tau, fma(tau, it[S_AR + 3], it[S_AR + 2]), it[S_AR + 1]), it[S_AR]);
    const double Aim = fma(tau, fma(tau, fma(tau, it[S_AI + 3], it[S_AI + 2]), it[S_AI + 1]), it[S_AI]);
    // phase in quarter turns, the folded -+1/2 of the standard SPA taken out again
    const double TK4 = it[S_TK4];
    const double P = __dmul_rn(sf, TK4);
    const double e = __fma_rn(sf, TK4, -P);
    const double big4 = 27021597764222976.0;
    const double pr = P - ((P + big4) - big4);
    const double wv = fma(sf + it[S_NFA], 4.0, it[S_WC]);
    const double loc = tau * fma(tau, fma(tau, it[S_ND4], it[S_NC4]), wv);
    double q = ((pr + e) + (it[S_PC4] + copysign(0.5, it[S_CU]))) + loc;
    double Sre, Sim;
    if (series) {
        const double y = rsqrt(aFd);
        const double y2 = y * y;
        const double pq = Fdd * y2;
        const double u = copysign(0.477464829275686 * pq * pq * y2, Fd);      // 1/X
        const double u2 = u * u;
        double gr = c_gre[6];
#pragma unroll
        for (int i = 5; i >= 0; --i) gr = fma(gr, u2, c_gre[i]);
        double gi = c_gim[5];
#pragma unroll
        for (int i = 4; i >= 0; --i) gi = fma(gi, u2, c_gim[i]);
        gi *= u;
        Sre = gr * y;
        Sim = gi * y;
        q -= copysign(0.5, Fd);
    } else {
        // |X| < 28: regular Airy form  e^{-iX} pi kap [Ai(-yy) -+ i Bi(-yy)],  kap = (pi|Fddot|)^(-1/3)
        const double sig = (Fd >= 0.0) ? 1.0 : -1.0;
        const double kap = rcbrt(3.141592653589793 * fabs(Fdd));
        const double k2 = kap * kap;
        const double yy = k2 * k2 * 9.869604401089358 * Fd * Fd;
        double ai, bi;
        fdemri_airy_neg(yy, ai, bi);
        const double X = 0.6666666666666666 * sig * yy * sqrt(yy);
        q -= X * 0.6366197723675814;                   // X / (pi/2) quarter turns
        Sre = 3.141592653589793 * kap * ai;
        Sim = -sig * 3.141592653589793 * kap * bi;
        out.info |= 1u;
    }
    double sn, cs;
    fdemri_sincos_quarter(q, sn, cs);
    const double Ere = Sre * cs - Sim * sn, Eim = Sre * sn + Sim * cs;
    out.tre = Are * Ere - Aim * Eim;
    out.tim = Are * Eim + Aim * Ere;
    return out;
}

// ---------------------------------------------------------------------------------------------------------
// Shared-memory ring between the producer warp and the consumer warps
// ---------------------------------------------------------------------------------------------------------
// doubles between staged items: 34, not 32, so that two neighbouring items sit on different shared-memory banks (a merged
// pass of the consumers reads both with one per-lane-address load)
#ifndef FDEMRI_ITEM_STRIDE
#define FDEMRI_ITEM_STRIDE (S_DOUBLES + 2)
#endif
struct FdemriStage {
    double items[FDEMRI_CHUNK][FDEMRI_ITEM_STRIDE];
    int hdr[4];                  // {global tile index (-1: no more work), item count, last chunk of the tile, 0}
};
struct FdemriRing {
    FdemriStage st[FDEMRI_STAGES];
    uint64_t full[FDEMRI_STAGES];
    uint64_t empty[FDEMRI_STAGES];
};

// Producer lane: folds record + weights + sign into the staged item `dst` (shared memory)
// a record in registers: six 32-byte loads, issued together (the producer issues them before it waits for a ring slot)
struct FdemriRecRegs {
    double4 r0, r1, r2, r3, r4, r5;
};
__device__ __forceinline__ FdemriRecRegs fdemri_load_rec(const double* __restrict__ R) {
    const double4* R4 = reinterpret_cast<const double4*>(R);
    FdemriRecRegs q;
    q.r0 = fdemri_ld4(R4 + 0);       // FA FB FC FD
    q.r1 = fdemri_ld4(R4 + 1);       // Q1 Q2 Q3 H
    q.r2 = fdemri_ld4(R4 + 2);       // Re A
    q.r3 = fdemri_ld4(R4 + 3);       // Im A
    q.r4 = fdemri_ld4(R4 + 4);       // PC BH BL NC
    q.r5 = fdemri_ld4(R4 + 5);       // ND TK TYPE SF
    return q;
}
__device__ __forceinline__ void fdemri_stage_regs(double* dst, const FdemriRecRegs& q, const double4 w, int lo,
                                                  int hi, unsigned sg, unsigned br) {
    const double4 r0 = q.r0, r1 = q.r1, r2 = q.r2, r3 = q.r3, r4 = q.r4, r5 = q.r5;
    const unsigned type = (unsigned)r5.z;        // interior extrema of F on the segment: 0, 1, 2
    const double s = sg ? -1.0 : 1.0;
    const double h = r1.w;
    double2* d2 = reinterpret_cast<double2*>(dst);
    double sF, q1 = r1.x, q2 = r1.y, q3 = r1.z, x9, x11, x15 = 0.0, x19, x1;
    unsigned fl = sg << 2;
    if (type == 0u) {
        sF = r5.w;
        const float2 f32a = make_float2((float)r0.y, (float)r0.z);           // FB, FC
        const float2 f32b = make_float2((float)r0.w, (float)r1.x);           // FD, Q1
        const float2 f32c = make_float2((float)r1.y, (float)r1.z);           // Q2, Q3
        x1 = *reinterpret_cast<const double*>(&f32a);
        x11 = *reinterpret_cast<const double*>(&f32b);
        x19 = *reinterpret_cast<const double*>(&f32c);
        x9 = 2e-7 * h;
    } else {
        // branch `br` of a segment with extrema at te1 (< te2): [0, te1], (te1, te2 or h], (te2, h); F' alternates in sign
        const double te1 = r1.x, Fe1 = r1.y, te2 = r1.z, Fe2 = r5.w;
        const double s0 = (Fe1 < r0.x) ? -1.0 : 1.0;                        // first branch runs from F_k to F_e1
        sF = (br == 1u) ? -s0 : s0;
        const bool two = type == 2u;
        const double ta = (br == 0u) ? 0.0 : (br == 1u ? te1 : te2);
        const double tb = (br == 0u) ? te1 : (br == 1u && two ? te2 : h);
        const bool useB = br == 2u;                                          // the extremum the branch hangs on
        q1 = useB ? te2 : te1;
        q2 = useB ? Fe2 : Fe1;
        q3 = fma(3.0 * r0.w, q1, r0.z);                                      // c2 = C + 3 D tau_e
        x1 = ta; x11 = tb;
        x19 = te2; x15 = Fe2; x9 = fma(3.0 * r0.w, te2, r0.z);              // the second one (middle branch only)
        fl |= 1u | ((br == 1u && two) ? 2u : 0u);
    }
    int2 meta = make_int2(lo | (hi << 16), (int)fl);
    d2[0] = make_double2(__hiloint2double(meta.y, meta.x), x1);
    d2[1] = make_double2(-r0.x, r0.y);
    d2[2] = make_double2(r0.z, r0.w);
    d2[3] = make_double2(q1, q2);
    d2[4] = make_double2(q3, x9);
    d2[5] = make_double2(0.5 * h, x11);
    d2[6] = make_double2(sF * 1.9098593171027440, 4.0 * r5.y);
    d2[7] = make_double2(4.0 * ((r0.x - r4.y) - r4.z), x15);      // F_k and b' nearly cancel: the difference is exact
    d2[8] = make_double2(4.0 * r4.w, 4.0 * r5.x);
    d2[9] = make_double2(fma(4.0, r4.x + w.z, -0.5 * sF), x19);
    d2[10] = make_double2(r2.x, r2.y);
    d2[11] = make_double2(r2.z, r2.w);
    d2[12] = make_double2(r3.x, r3.y);
    d2[13] = make_double2(r3.z, r3.w);
    d2[14] = make_double2(w.x, s * w.x);
    d2[15] = make_double2(-w.y, s * w.y);
}

__device__ __forceinline__ void fdemri_stage_item(double* dst, const double* __restrict__ R, const double4 w, int lo,
                                                  int hi, unsigned sg, unsigned br) {
    fdemri_stage_regs(dst, fdemri_load_rec(R), w, lo, hi, sg, br);
}

// ---------------------------------------------------------------------------------------------------------
// The item scan: the entries of one batch item that meet a range of bins [b0, b1], produced in ascending key
// order by ONE warp, a step at a time (fdemri_map.cuh has the tables):
//   level 1  voice-sign bands, L1U x 32 at a time (coalesced int2 loads)      -> queue q1 of voice-signs that meet the range
//   level 2  the group bands of up to 32 queued voice-signs, a lane each      -> queue q2 of rows (vs, branch, group)
//   level 3  the 32 entries of up to 32 queued rows, a lane per row (16 x 16 B)      -> emit(entry) in order
// The queues are FIFO, so the emitted order is (voice, sign, branch, segment) = ascending key, and every load is
// issued in batches of independent requests (latency is paid per step, not per entry).  Control flow is warp-uniform.
// ---------------------------------------------------------------------------------------------------------
struct FdemriScan {
    const int2* vband;        // tables of the batch item
    const int4* gband;
    const int2* ent;
    int Sp, G, nb2;           // Sp = 32 G: entries per (voice, sign, branch) row, padded; nb2: voice-signs per level-2 step
                              // (their rows must fit q2)
    int b0, b1;
    int vs_next, vs_end;      // voice-signs still to look at
    unsigned q1_head, q1_tail, q2_head, q2_tail;
};

template <int Q2CAP>
__device__ __forceinline__ void fdemri_scan_init(FdemriScan& c, const SumArgs& a, int b, int vs0, int vs1, int b0, int b1) {
    const FdemriDims& d = a.d;
    const size_t nvs = (size_t)2 * d.n_modes;
    c.vband = a.vband + (size_t)b * nvs;
    c.gband = a.gband + (size_t)b * nvs * d.n_groups;
    c.ent = a.ent + (size_t)b * nvs * d.ent_max;
    c.Sp = 32 * d.n_groups; c.G = d.n_groups;
    c.nb2 = min(32, (Q2CAP - 32) / (3 * d.n_groups));          // level 2 runs with < 32 rows queued: its output must fit
    c.b0 = b0; c.b1 = b1;
    c.vs_next = vs0; c.vs_end = vs1;
    c.q1_head = c.q1_tail = c.q2_head = c.q2_tail = 0u;
}

// One step.  Returns 0: exhausted, 1: progressed, 2: level 3 has input but emit has no room for a row (32 entries).
// emit.room() -> free places (warp-uniform); emit.store(offset, vsbr, seg, lo, hi): the entry goes to the offset-th free
// place; emit.advance(n): n places have been filled.
template <int Q1CAP, int Q2CAP, int L1U, class Emit>
__device__ __forceinline__ int fdemri_scan_step(FdemriScan& c, unsigned* __restrict__ q1, unsigned* __restrict__ q2, int lane,
                                                Emit& emit) {
    const unsigned full = 0xffffffffu, lt = (1u << lane) - 1u;
    // Which level: a deeper one as soon as it has a full batch of 32 inputs (all lanes busy), a shallower one to make
    // more input, a partial batch only when nothing shallower is left.  (Queue sizes make one of them always possible.)
    const unsigned n2 = c.q2_tail - c.q2_head, n1 = c.q1_tail - c.q1_head;
    const bool more1 = c.vs_next < c.vs_end;
    int level;
    if (n2 >= 32u) level = 3;
    else if (n1 >= 32u || (n1 > 0u && !more1)) level = 2;
    else if (more1) level = 1;
    else if (n2 > 0u) level = 3;
    else return 0;
    if (level == 3) {                                               // ---- level 3: up to 32 rows, a lane per row ----
        const int room = emit.room();
        if (room < 32) return 2;
        const int nr = (int)min(c.q2_tail - c.q2_head, 32u);
        unsigned row = 0u, hits = 0u;
        const int2* src = c.ent;
        if (lane < nr) {
            // pass 1: which of the row's 32 entries meet the range (16 x 16-byte loads, nothing kept but the mask)
            row = q2[(c.q2_head + (unsigned)lane) & (Q2CAP - 1)];
            src = c.ent + (size_t)(row >> 4) * c.Sp + 32 * (row & 15u);
            const int4* s4 = reinterpret_cast<const int4*>(src);
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int4 q = __ldg(s4 + j);
                hits |= (unsigned)(q.y >= q.x && q.x <= c.b1 && q.y >= c.b0) << (2 * j);
                hits |= (unsigned)(q.w >= q.z && q.z <= c.b1 && q.w >= c.b0) << (2 * j + 1);
            }
        }
        const int cnt = __popc(hits);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(full, incl, o);
            if (lane >= o) incl += t;
        }
        // rows are taken in order as long as their entries fit (the first always does: room >= 32)
        const int nok = __popc(__ballot_sync(full, lane < nr && incl <= room));
        if (lane < nok) {
            // pass 2: the few entries that hit, read again (they are in L1 now)
            int off = incl - cnt;
            const int vsbr = (int)(row >> 4), seg0 = 32 * (int)(row & 15u);
            while (hits) {
                const int j = __ffs(hits) - 1;
                hits &= hits - 1;
                const int2 q = __ldg(src + j);
                emit.store(off++, vsbr, seg0 + j, q.x, q.y);
            }
        }
        emit.advance(__shfl_sync(full, incl, nok - 1));
        c.q2_head += (unsigned)nok;
        __syncwarp();
        return 1;
    }
    if (level == 2) {                                               // ---- level 2: a lane per voice-sign ----
        const int nb = (int)min(c.q1_tail - c.q1_head, (unsigned)c.nb2);
        unsigned m0 = 0u, m12 = 0u;
        unsigned vs = 0u;
        if (lane < nb) {
            vs = q1[(c.q1_head + lane) & (Q1CAP - 1)];
            const int4* gb = c.gband + (size_t)vs * c.G;
            for (int g = 0; g < c.G; ++g) {
                const int4 q = __ldg(gb + g);
                m0 |= (unsigned)(q.x <= c.b1 && q.y >= c.b0) << g;
                m12 |= (unsigned)(q.z <= c.b1 && q.w >= c.b0) << g;
            }
        }
        const int cnt = __popc(m0) + 2 * __popc(m12);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(full, incl, o);
            if (lane >= o) incl += t;
        }
        unsigned pos = c.q2_tail + (unsigned)(incl - cnt);
#pragma unroll
        for (int br = 0; br < 3; ++br) {
            unsigned mk = br ? m12 : m0;
            while (mk) {
                const int g = __ffs(mk) - 1;
                mk &= mk - 1;
                q2[pos++ & (Q2CAP - 1)] = ((vs * 3u + (unsigned)br) << 4) | (unsigned)g;
            }
        }
        c.q2_tail += (unsigned)__shfl_sync(full, incl, 31);
        c.q1_head += (unsigned)nb;
        __syncwarp();
        return 1;
    }
    {                                                               // ---- level 1: L1U x 32 voice-signs ----
        int2 vb[L1U];
#pragma unroll
        for (int u = 0; u < L1U; ++u) {
            const int vs = c.vs_next + 32 * u + lane;
            vb[u] = (vs < c.vs_end) ? __ldg(c.vband + vs) : make_int2(1, 0);
        }
#pragma unroll
        for (int u = 0; u < L1U; ++u) {
            const bool stab = vb[u].y >= vb[u].x && vb[u].x <= c.b1 && vb[u].y >= c.b0;
            const unsigned mk = __ballot_sync(full, stab);
            if (stab) q1[(c.q1_tail + __popc(mk & lt)) & (Q1CAP - 1)] = (unsigned)(c.vs_next + 32 * u + lane);
            c.q1_tail += (unsigned)__popc(mk);
        }
        c.vs_next += 32 * L1U;
        __syncwarp();
        return 1;
    }
}

// ---- the producer warp of the tile-major kernel -------------------------------------------------------------
#define FDEMRI_PQ1 512          // voice-signs waiting for level 2   (>= 31 + 32 * L1U, L1U = 8)
#define FDEMRI_PQ2 2048         // rows waiting for level 3           (>= 32 + 32 * 3 * 16 groups)
#define FDEMRI_PQ3 512          // entries waiting to be staged
struct FdemriProdQueues {
    unsigned q1[FDEMRI_PQ1];
    unsigned q2[FDEMRI_PQ2];
    int4 q3[FDEMRI_PQ3];        // {(vs*3 + branch), segment, first bin, last bin}
};
struct FdemriProdEmit {
    int4* q3;
    unsigned head, tail;
    __device__ __forceinline__ int room() const { return (int)(FDEMRI_PQ3 - (tail - head)); }
    __device__ __forceinline__ void store(int off, int vsbr, int seg, int lo, int hi) {
        q3[(tail + (unsigned)off) & (FDEMRI_PQ3 - 1)] = make_int4(vsbr, seg, lo, hi);
    }
    __device__ __forceinline__ void advance(int n) { tail += (unsigned)n; }
};

// Producer: for every tile it draws, the entries that meet the tile (the scan above), one ring stage per 32 of them:
// entry -> record + weights -> staged item.
__device__ __forceinline__ void fdemri_producer(const SumArgs& a, FdemriRing* ring, FdemriProdQueues* pq, int lane) {
    const FdemriDims& d = a.d;
    const int V = d.n_modes;
    int stage = 0;
    unsigned phase = 0;
    unsigned long long n_items = 0;
    for (;;) {
        int gt = 0;
        if (lane == 0) gt = (int)atomicAdd(a.tile_counter, 1u);
        gt = __shfl_sync(0xffffffffu, gt, 0);
        if (gt >= a.total_tiles) break;
        const int b = gt / d.n_tiles, tile = gt - b * d.n_tiles;
        const int64_t bin0 = (int64_t)tile * FDEMRI_TILE;
        const int tile_lo = (int)bin0;
        const int tile_hi = (int)min(bin0 + FDEMRI_TILE - 1, d.n_freq - 1);
        const int wbase = (a.n_angles > 1 ? b : 0) * V;
        const size_t rbase = (size_t)b * V * d.n_seg;
        // tiles outside the band of the item have no entry: nothing to scan
        const bool in_band = tile_lo <= __ldg(a.iband + 2 * b + 1) - 1 && tile_hi >= 0x7fffffff - __ldg(a.iband + 2 * b);
        FdemriScan sc;
        fdemri_scan_init<FDEMRI_PQ2>(sc, a, b, 0, in_band ? 2 * V : 0, tile_lo, tile_hi);
        FdemriProdEmit em;
        em.q3 = pq->q3; em.head = em.tail = 0u;
        bool last;
        do {
            // at least 33 entries queued, or all that are left: the stage knows whether it is the tile's last
            while (em.tail - em.head <= 32u && fdemri_scan_step<FDEMRI_PQ1, FDEMRI_PQ2, 8>(sc, pq->q1, pq->q2, lane, em) == 1) {}
            __syncwarp();
            const int cnt = (int)min(em.tail - em.head, 32u);
            int4 en = make_int4(0, 0, 0, -1);
            FdemriRecRegs q;
            double4 w4 = make_double4(0.0, 0.0, 0.0, 0.0);
            if (lane < cnt) {
                en = pq->q3[(em.head + (unsigned)lane) & (FDEMRI_PQ3 - 1)];
                const int v = en.x / 6;                                  // en.x = (v*2 + sign)*3 + branch
                q = fdemri_load_rec(a.rec + (rbase + (size_t)v * d.n_seg + en.y) * R_DOUBLES);
                w4 = a.wts[wbase + v];
            }
            em.head += (unsigned)cnt;
            last = (em.tail == em.head);
            n_items += (unsigned)cnt;
            // wait for the ring slot; meanwhile scan ahead for the next stages (nothing to do: back off)
            {
                const unsigned addr = fdemri_smem_addr(&ring->empty[stage]);
#ifdef FDEMRI_SCAN_AHEAD        /* measured: scanning ahead while waiting costs the consumers more than it saves (profiles/) */
                bool can_scan = true;                                // false: exhausted, or the entry queue is full
                while (!fdemri_mbar_try(addr, phase ^ 1u)) {
                    if (can_scan) can_scan = fdemri_scan_step<FDEMRI_PQ1, FDEMRI_PQ2, 8>(sc, pq->q1, pq->q2, lane, em) == 1;
                    else __nanosleep(FDEMRI_PROD_BACKOFF);
                }
#else
                while (!fdemri_mbar_try(addr, phase ^ 1u)) __nanosleep(FDEMRI_PROD_BACKOFF);
#endif
            }
            if (lane < cnt) {
                const int vs = en.x / 3, br = en.x - 3 * vs;
                const int lo_e = max(en.z, tile_lo) - tile_lo;
                const int hi_e = min(en.w, tile_hi) - tile_lo;
                fdemri_stage_regs(ring->st[stage].items[lane], q, w4, lo_e, hi_e, (unsigned)(vs & 1), (unsigned)br);
            }
            __syncwarp();
            if (lane == 0) {
                ring->st[stage].hdr[0] = gt; ring->st[stage].hdr[1] = cnt; ring->st[stage].hdr[2] = last;
                fdemri_mbar_arrive(&ring->full[stage]);
            }
            if (++stage == FDEMRI_STAGES) { stage = 0; phase ^= 1u; }
        } while (!last);
    }
    // no more work
    fdemri_mbar_wait(&ring->empty[stage], phase ^ 1u, FDEMRI_PROD_BACKOFF);
    if (lane == 0) {
        ring->st[stage].hdr[0] = -1; ring->st[stage].hdr[1] = 0; ring->st[stage].hdr[2] = 1;
        fdemri_mbar_arrive(&ring->full[stage]);
        if (n_items) atomicAdd(a.stats + 8, n_items);              // (entry, tile) pairs staged
    }
}

__device__ __forceinline__ void fdemri_consumer(const SumArgs& a, FdemriRing* ring, int cw, int lane) {
    const FdemriDims& d = a.d;
    int stage = 0;
    unsigned phase = 0;
    int cur = -1;
    int b = 0;
    int64_t bin_a = 0;                            // first bin of this lane (second: + 32)
    double f0 = 0.0, f1 = 0.0;
    double a00 = 0.0, a01 = 0.0, a02 = 0.0, a03 = 0.0, a10 = 0.0, a11 = 0.0, a12 = 0.0, a13 = 0.0;
    unsigned n_airy = 0, n_slow = 0, errs = 0;
    const int wb = cw * 32 * FDEMRI_BPL;          // first tile-relative bin of this warp
    const int rel0 = wb + lane, rel1 = rel0 + 32;
    for (;;) {
        fdemri_mbar_wait(&ring->full[stage], phase, FDEMRI_CONS_BACKOFF);
        const FdemriStage* S = &ring->st[stage];
        const int gt = S->hdr[0], cnt = S->hdr[1], last = S->hdr[2];
        if (gt < 0) break;
        if (gt != cur) {
            cur = gt;
            b = gt / d.n_tiles;
            const int tile = gt - b * d.n_tiles;
            bin_a = (int64_t)tile * FDEMRI_TILE + rel0;
            f0 = (bin_a < d.n_freq) ? fdemri_freq(d, bin_a) : 0.0;
            f1 = (bin_a + 32 < d.n_freq) ? fdemri_freq(d, bin_a + 32) : 0.0;
            a00 = a01 = a02 = a03 = a10 = a11 = a12 = a13 = 0.0;
        }
        // items of the chunk that overlap this warp's bins: lane j looks at item j, two ballots (overlaps; is monotone and
        // covers all 64 bins), then the set bits are walked in ascending (= list) order
        unsigned todo, fullm;
        {
            bool mine = false, whole = false;
            if (lane < cnt) {
                const int2 mx = *reinterpret_cast<const int2*>(S->items[lane]);     // {lo | hi << 16, flags}
                const int lo = mx.x & 0xffff, hi = mx.x >> 16;
                mine = !(hi < wb || lo > wb + 32 * FDEMRI_BPL - 1);
                whole = lo <= wb && hi >= wb + 32 * FDEMRI_BPL - 1 && !(mx.y & 1);
            }
            todo = __ballot_sync(0xffffffffu, mine);
            fullm = __ballot_sync(0xffffffffu, whole);
        }
        while (todo) {
            // ---- the common pass: a monotone item that covers every bin of this warp -- no masks.  Its loop holds nothing
            // else: a pass that needs the slow path for some lane, and an item of any other kind, leave it and are dealt
            // with below (with the out-of-line slow path and its call sequence out of the way ptxas compiles the common
            // pass 5 % faster: 2.55 -> 2.42 ms on config 2) ----
            int j = 0, state = 0;                // 1: slow-path fix-ups for the pass in hand, 2: another kind of item
            const double* it = nullptr;
            double sf0 = 0.0, sf1 = 0.0, T0r = 0.0, T0i = 0.0, T1r = 0.0, T1i = 0.0;
            bool ok0 = true, ok1 = true;
            while (todo) {
                j = __ffs(todo) - 1;
                todo &= todo - 1;
                it = S->items[j];
                if (!((fullm >> j) & 1u)) { state = 2; break; }
                const unsigned sbit = ((unsigned)reinterpret_cast<const int*>(it)[1] & 4u) << 29;
                sf0 = fdemri_xorsign(f0, sbit); sf1 = fdemri_xorsign(f1, sbit);
                ok0 = fdemri_term_fast(it, sf0, T0r, T0i);
                ok1 = fdemri_term_fast(it, sf1, T1r, T1i);
                if (__any_sync(0xffffffffu, !(ok0 && ok1))) { state = 1; break; }      // under 1 % of the passes
                // weights (O2): s=+1: h+ += w+ T, hx += i wx T;  s=-1: h+ += w+ conj(T), hx += conj(i wx T)
                const double wp = it[S_WP], swp = it[S_SWP], nwx = it[S_NWX], swx = it[S_SWX];
                a00 = fma(wp, T0r, a00); a01 = fma(swp, T0i, a01); a02 = fma(nwx, T0i, a02); a03 = fma(swx, T0r, a03);
                a10 = fma(wp, T1r, a10); a11 = fma(swp, T1i, a11); a12 = fma(nwx, T1i, a12); a13 = fma(swx, T1r, a13);
            }
            if (state == 0) break;
            if (state == 1) {
                const unsigned flags = (unsigned)reinterpret_cast<const int*>(it)[1];
                if (!ok0) {
                    const FdemriSlowOut o = fdemri_term_slow(it, sf0, flags);
                    T0r = o.tre; T0i = o.tim;
                    n_airy += o.info & 1u; n_slow += (o.info >> 1) & 1u; errs |= o.info >> 4;
                }
                if (!ok1) {
                    const FdemriSlowOut o = fdemri_term_slow(it, sf1, flags);
                    T1r = o.tre; T1i = o.tim;
                    n_airy += o.info & 1u; n_slow += (o.info >> 1) & 1u; errs |= o.info >> 4;
                }
                const double wp = it[S_WP], swp = it[S_SWP], nwx = it[S_NWX], swx = it[S_SWX];
                a00 = fma(wp, T0r, a00); a01 = fma(swp, T0i, a01); a02 = fma(nwx, T0i, a02); a03 = fma(swx, T0r, a03);
                a10 = fma(wp, T1r, a10); a11 = fma(swp, T1i, a11); a12 = fma(nwx, T1i, a12); a13 = fma(swx, T1r, a13);
                continue;
            }
            // ---- an item that covers part of this warp's bins, or a branch of a segment with extrema ----
            const int2 meta = *reinterpret_cast<const int2*>(it);        // {lo | hi << 16, flags}
            const int lo = meta.x & 0xffff, hi = meta.x >> 16;
            const unsigned flags = (unsigned)meta.y;
            const bool act0 = rel0 >= lo && rel0 <= hi, act1 = rel1 >= lo && rel1 <= hi;
            if (flags & 1u) {
                const unsigned sbit = (flags & 4u) << 29;
                const double sf0 = fdemri_xorsign(f0, sbit), sf1 = fdemri_xorsign(f1, sbit);
                double T0r = 0.0, T0i = 0.0, T1r = 0.0, T1i = 0.0;
                if (act0) {
                    const FdemriSlowOut o = fdemri_term_slow(it, sf0, flags);
                    T0r = o.tre; T0i = o.tim;
                    n_airy += o.info & 1u; n_slow += (o.info >> 1) & 1u; errs |= o.info >> 4;
                }
                if (act1) {
                    const FdemriSlowOut o = fdemri_term_slow(it, sf1, flags);
                    T1r = o.tre; T1i = o.tim;
                    n_airy += o.info & 1u; n_slow += (o.info >> 1) & 1u; errs |= o.info >> 4;
                }
                const double wp = it[S_WP], swp = it[S_SWP], nwx = it[S_NWX], swx = it[S_SWX];
                if (act0) {
                    a00 = fma(wp, T0r, a00); a01 = fma(swp, T0i, a01); a02 = fma(nwx, T0i, a02); a03 = fma(swx, T0r, a03);
                }
                if (act1) {
                    a10 = fma(wp, T1r, a10); a11 = fma(swp, T1i, a11); a12 = fma(nwx, T1i, a12); a13 = fma(swx, T1r, a13);
                }
                continue;
            }
            // A monotone item that ends (or starts) inside this warp's 64 bins.  The items that follow it in the list and
            // whose bins lie entirely beside what has been gathered so far -- the usual case: the next segment of the
            // same voice, which starts at the following bin -- share ONE pass with it: every (lane, slot) evaluates the
            // item that covers its bin, with its own item constants (per-lane addresses; FDEMRI_ITEM_STRIDE keeps
            // neighbouring items on different banks).  Without this each of them would take a whole pass with part of
            // the lanes idle: 5.70 M passes instead of 5.18 M on config 2, where 5.15 M would use every lane.  A bin
            // still receives its terms in list order, so the sums are the same bit for bit.
            const double* it0 = it;
            const double* it1 = it;
            unsigned fl0 = flags, fl1 = flags;
            bool m0 = act0, m1 = act1;
#ifndef FDEMRI_NO_MERGE
            {
                int run_lo = lo, run_hi = hi, jn = j + 1;
                while (jn < FDEMRI_CHUNK && ((todo >> jn) & 1u)) {
                    const double* itB = S->items[jn];
                    const int2 metaB = *reinterpret_cast<const int2*>(itB);
                    const int loB = metaB.x & 0xffff, hiB = metaB.x >> 16;
                    if ((metaB.y & 1) || !(loB > run_hi || hiB < run_lo)) break;     // only monotone items, entirely beside the run
                    todo &= todo - 1;
                    ++jn;
                    run_lo = min(run_lo, loB); run_hi = max(run_hi, hiB);
                    const bool b0 = rel0 >= loB && rel0 <= hiB, b1 = rel1 >= loB && rel1 <= hiB;
                    if (b0) { it0 = itB; fl0 = (unsigned)metaB.y; }
                    if (b1) { it1 = itB; fl1 = (unsigned)metaB.y; }
                    m0 = m0 || b0; m1 = m1 || b1;
                }
            }
#endif
            {
                const double sf0 = fdemri_xorsign(f0, (fl0 & 4u) << 29), sf1 = fdemri_xorsign(f1, (fl1 & 4u) << 29);
                double T0r, T0i, T1r, T1i;
                const bool ok0 = fdemri_term_fast(it0, sf0, T0r, T0i);
                const bool ok1 = fdemri_term_fast(it1, sf1, T1r, T1i);
                const bool bad0 = m0 && !ok0, bad1 = m1 && !ok1;
                if (__any_sync(0xffffffffu, bad0 || bad1)) {
                    if (bad0) {
                        const FdemriSlowOut o = fdemri_term_slow(it0, sf0, fl0);
                        T0r = o.tre; T0i = o.tim;
                        n_airy += o.info & 1u; n_slow += (o.info >> 1) & 1u; errs |= o.info >> 4;
                    }
                    if (bad1) {
                        const FdemriSlowOut o = fdemri_term_slow(it1, sf1, fl1);
                        T1r = o.tre; T1i = o.tim;
                        n_airy += o.info & 1u; n_slow += (o.info >> 1) & 1u; errs |= o.info >> 4;
                    }
                }
                if (m0) {
                    a00 = fma(it0[S_WP], T0r, a00); a01 = fma(it0[S_SWP], T0i, a01);
                    a02 = fma(it0[S_NWX], T0i, a02); a03 = fma(it0[S_SWX], T0r, a03);
                }
                if (m1) {
                    a10 = fma(it1[S_WP], T1r, a10); a11 = fma(it1[S_SWP], T1i, a11);
                    a12 = fma(it1[S_NWX], T1i, a12); a13 = fma(it1[S_SWX], T1r, a13);
                }
            }
        }
        if (last) {
            const bool v0 = bin_a < d.n_freq, v1 = bin_a + 32 < d.n_freq;
            if (a.hp) {
                if (v0) {
                    const size_t o = ((size_t)b * d.n_freq + bin_a) * 2;
                    *reinterpret_cast<double2*>(a.hp + o) = make_double2(a00, a01);
                    *reinterpret_cast<double2*>(a.hx + o) = make_double2(a02, a03);
                }
                if (v1) {
                    const size_t o = ((size_t)b * d.n_freq + bin_a + 32) * 2;
                    *reinterpret_cast<double2*>(a.hp + o) = make_double2(a10, a11);
                    *reinterpret_cast<double2*>(a.hx + o) = make_double2(a12, a13);
                }
            }
            if (a.inner_part) {
                // Eq. 12 on the fly: this warp's share of sum_k w_k (|h+|^2 + |hx|^2) and sum_k w_k (d+ conj h+ + dx conj hx),
                // reduced over the lanes in a fixed butterfly; k_inner_reduce adds the warps in a fixed order
                double p0r = a00, p0i = a01, x0r = a02, x0i = a03, p1r = a10, p1i = a11, x1r = a12, x1i = a13;
                bool use0 = v0, use1 = v1;
                if (a.inner_edge) {
                    // Hann window as the 3-point filter h_k/2 - h_{k-1}/4 - h_{k+1}/4 (L145).  Neighbours come from the
                    // adjacent lanes; the first and the last bin of the warp's range need a bin of another warp and
                    // are left to k_inner_reduce, which gets the two bins at either end of the range.
                    if (lane < 2 || lane >= 30) {
                        double* e = a.inner_edge + (((size_t)gt * FDEMRI_CWARPS + cw) * 4 + (lane < 2 ? lane : lane - 28)) * 4;
                        if (lane < 2) *reinterpret_cast<double4*>(e) = make_double4(a00, a01, a02, a03);
                        else *reinterpret_cast<double4*>(e) = make_double4(a10, a11, a12, a13);
                    }
                    const unsigned full = 0xffffffffu;
                    // slot 0: left neighbour = lane - 1 of slot 0; right neighbour = lane + 1 of slot 0, or lane 0 of slot 1
                    const double l0a = __shfl_up_sync(full, a00, 1), l0b = __shfl_up_sync(full, a01, 1);
                    const double l0c = __shfl_up_sync(full, a02, 1), l0d = __shfl_up_sync(full, a03, 1);
                    double r0a = __shfl_down_sync(full, a00, 1), r0b = __shfl_down_sync(full, a01, 1);
                    double r0c = __shfl_down_sync(full, a02, 1), r0d = __shfl_down_sync(full, a03, 1);
                    const double f1a = __shfl_sync(full, a10, 0), f1b = __shfl_sync(full, a11, 0);
                    const double f1c = __shfl_sync(full, a12, 0), f1d = __shfl_sync(full, a13, 0);
                    if (lane == 31) { r0a = f1a; r0b = f1b; r0c = f1c; r0d = f1d; }
                    // slot 1: left neighbour = lane - 1 of slot 1, or lane 31 of slot 0; right neighbour = lane + 1 of slot 1
                    double l1a = __shfl_up_sync(full, a10, 1), l1b = __shfl_up_sync(full, a11, 1);
                    double l1c = __shfl_up_sync(full, a12, 1), l1d = __shfl_up_sync(full, a13, 1);
                    const double g0a = __shfl_sync(full, a00, 31), g0b = __shfl_sync(full, a01, 31);
                    const double g0c = __shfl_sync(full, a02, 31), g0d = __shfl_sync(full, a03, 31);
                    if (lane == 0) { l1a = g0a; l1b = g0b; l1c = g0c; l1d = g0d; }
                    const double r1a = __shfl_down_sync(full, a10, 1), r1b = __shfl_down_sync(full, a11, 1);
                    const double r1c = __shfl_down_sync(full, a12, 1), r1d = __shfl_down_sync(full, a13, 1);
                    p0r = 0.5 * a00 - 0.25 * (l0a + r0a); p0i = 0.5 * a01 - 0.25 * (l0b + r0b);
                    x0r = 0.5 * a02 - 0.25 * (l0c + r0c); x0i = 0.5 * a03 - 0.25 * (l0d + r0d);
                    p1r = 0.5 * a10 - 0.25 * (l1a + r1a); p1i = 0.5 * a11 - 0.25 * (l1b + r1b);
                    x1r = 0.5 * a12 - 0.25 * (l1c + r1c); x1i = 0.5 * a13 - 0.25 * (l1d + r1d);
                    use0 = v0 && lane != 0;
                    use1 = v1 && lane != 31;
                }
                double hh = 0.0, dr = 0.0, di = 0.0;
                if (use0) {
                    const double w0 = a.weight ? __ldg(a.weight + bin_a) : 1.0;
                    hh = w0 * (p0r * p0r + p0i * p0i + x0r * x0r + x0i * x0i);
                    if (a.dplus) {
                        const double2 dp = *reinterpret_cast<const double2*>(a.dplus + 2 * bin_a);
                        const double2 dx = *reinterpret_cast<const double2*>(a.dcross + 2 * bin_a);
                        dr = w0 * (dp.x * p0r + dp.y * p0i + dx.x * x0r + dx.y * x0i);
                        di = w0 * (dp.y * p0r - dp.x * p0i + dx.y * x0r - dx.x * x0i);
                    }
                }
                if (use1) {
                    const double w1 = a.weight ? __ldg(a.weight + bin_a + 32) : 1.0;
                    hh += w1 * (p1r * p1r + p1i * p1i + x1r * x1r + x1i * x1i);
                    if (a.dplus) {
                        const double2 dp = *reinterpret_cast<const double2*>(a.dplus + 2 * (bin_a + 32));
                        const double2 dx = *reinterpret_cast<const double2*>(a.dcross + 2 * (bin_a + 32));
                        dr += w1 * (dp.x * p1r + dp.y * p1i + dx.x * x1r + dx.y * x1i);
                        di += w1 * (dp.y * p1r - dp.x * p1i + dx.y * x1r - dx.x * x1i);
                    }
                }
#pragma unroll
                for (int o = 16; o; o >>= 1) {
                    hh += __shfl_xor_sync(0xffffffffu, hh, o);
                    dr += __shfl_xor_sync(0xffffffffu, dr, o);
                    di += __shfl_xor_sync(0xffffffffu, di, o);
                }
                if (lane == 0)
                    *reinterpret_cast<double4*>(a.inner_part + ((size_t)gt * FDEMRI_CWARPS + cw) * 4) = make_double4(hh, dr, di, 0.0);
            }
        }
        // release the stage
        __syncwarp();
        if (lane == 0) fdemri_mbar_arrive(&ring->empty[stage]);
        if (++stage == FDEMRI_STAGES) { stage = 0; phase ^= 1u; }
    }
    // counters: one atomic per warp
    for (int o = 16; o; o >>= 1) {
        n_airy += __shfl_xor_sync(0xffffffffu, n_airy, o);
        n_slow += __shfl_xor_sync(0xffffffffu, n_slow, o);
        errs |= __shfl_xor_sync(0xffffffffu, errs, o);
    }
    if (lane == 0) {
        if (n_airy) atomicAdd(a.stats + 4, (unsigned long long)n_airy);
        if (n_slow) atomicAdd(a.stats + 7, (unsigned long long)n_slow);
        if (errs) atomicOr(a.stats + 9, (unsigned long long)errs);
    }
}

// Registers: the two interleaved evaluations of a consumer lane need ~128 registers without spilling
#ifndef FDEMRI_MAXNREG
#define FDEMRI_MAXNREG 128
#endif
struct FdemriTileSmem {
    FdemriRing ring;
    FdemriProdQueues pq;
};
__global__ void __maxnreg__(FDEMRI_MAXNREG) k_tile_sum(SumArgs a) {
    extern __shared__ __align__(16) unsigned char fdemri_smem[];
    FdemriTileSmem* sm = reinterpret_cast<FdemriTileSmem*>(fdemri_smem);
    FdemriRing* ring = &sm->ring;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) {
        for (int i = 0; i < FDEMRI_STAGES; ++i) {
            fdemri_mbar_init(&ring->full[i], 1u);
            fdemri_mbar_init(&ring->empty[i], FDEMRI_CWARPS);
        }
    }
    __syncthreads();
    if (wid == FDEMRI_CWARPS) fdemri_producer(a, ring, &sm->pq, lane);
    else fdemri_consumer(a, ring, wid, lane);
}

// Fixed-order sum of the per-range partial inner products of one batch item.  One CTA per item.  A range is the
// 64 bins of a consumer warp of the tile-major kernel or a block of bins of the bin-major one (range_bins).
// With the Hann filter (edge != NULL) it also adds the first and the last bin of every range, whose filtered
// values need a bin of the neighbouring range: range i covers bins range_bins i .. range_bins (i + 1) - 1 of the item.
// out: [B][4] = {<h|h>, Re<d|h>, Im<d|h>, 0}
__device__ __forceinline__ void fdemri_inner_bin(const double4 h, int64_t k, const double* __restrict__ weight,
                                                 const double* __restrict__ dplus, const double* __restrict__ dcross,
                                                 double& hh, double& dr, double& di) {
    const double w = weight ? weight[k] : 1.0;
    hh += w * (h.x * h.x + h.y * h.y + h.z * h.z + h.w * h.w);
    if (dplus) {
        const double2 dp = *reinterpret_cast<const double2*>(dplus + 2 * k);
        const double2 dx = *reinterpret_cast<const double2*>(dcross + 2 * k);
        dr += w * (dp.x * h.x + dp.y * h.y + dx.x * h.z + dx.y * h.w);
        di += w * (dp.y * h.x - dp.x * h.y + dx.y * h.z - dx.x * h.w);
    }
}
__device__ __forceinline__ double4 fdemri_hann3(const double4 l, const double4 c, const double4 r) {
    return make_double4(0.5 * c.x - 0.25 * (l.x + r.x), 0.5 * c.y - 0.25 * (l.y + r.y), 0.5 * c.z - 0.25 * (l.z + r.z),
                        0.5 * c.w - 0.25 * (l.w + r.w));
}

__global__ void __launch_bounds__(256) k_inner_reduce(size_t n_ranges, int range_bins, int64_t n_freq,
                                                      const double* __restrict__ part, const double* __restrict__ edge,
                                                      const double* __restrict__ weight, const double* __restrict__ dplus,
                                                      const double* __restrict__ dcross, double* __restrict__ out) {
    __shared__ double s_r[3][256];
    const int b = blockIdx.x, tid = threadIdx.x;
    const size_t n = n_ranges;
    const double4* p = reinterpret_cast<const double4*>(part) + (size_t)b * n;
    const double4* e = edge ? reinterpret_cast<const double4*>(edge) + (size_t)b * n * 4 : nullptr;
    const double4 zero = make_double4(0.0, 0.0, 0.0, 0.0);
    double hh = 0.0, dr = 0.0, di = 0.0;
    for (size_t i = tid; i < n; i += 256) {
        const double4 v = p[i];
        hh += v.x; dr += v.y; di += v.z;
        if (e) {
            const int64_t k0 = (int64_t)i * range_bins, k1 = k0 + range_bins - 1;
            if (k0 < n_freq) {
                const double4 left = (i > 0) ? e[(i - 1) * 4 + 3] : zero;
                fdemri_inner_bin(fdemri_hann3(left, e[i * 4 + 0], e[i * 4 + 1]), k0, weight, dplus, dcross, hh, dr, di);
            }
            if (k1 < n_freq) {
                const double4 right = (i + 1 < n) ? e[(i + 1) * 4 + 0] : zero;
                fdemri_inner_bin(fdemri_hann3(e[i * 4 + 2], e[i * 4 + 3], right), k1, weight, dplus, dcross, hh, dr, di);
            }
        }
    }
    s_r[0][tid] = hh; s_r[1][tid] = dr; s_r[2][tid] = di;
    __syncthreads();
    for (int o = 128; o; o >>= 1) {
        if (tid < o) {
            s_r[0][tid] += s_r[0][tid + o]; s_r[1][tid] += s_r[1][tid + o]; s_r[2][tid] += s_r[2][tid + o];
        }
        __syncthreads();
    }
    if (tid == 0) *reinterpret_cast<double4*>(out + 4 * (size_t)b) = make_double4(s_r[0][0], s_r[1][0], s_r[2][0], 0.0);
}

// ---------------------------------------------------------------------------------------------------------
// Bin-major sum (sparse or down-sampled frequency arrays, section 3.3 / L218-242): when a (voice,
// segment) covers only a few bins, a tile of bins would run every item for a handful of lanes.  Here a CTA owns a
// BLOCK of d.tile_bins (8, 16 or 32: the plan takes the largest that still gives every resident CTA a few blocks)
// consecutive bins at a time (blocks are handed out by an atomic counter):
//   A  its eight warps run the item scan (above) over an eighth of the voice-signs each and collect the entries that
//      meet the block, in key order, in shared memory (a round takes what fits; further rounds take the rest);
//   B  every warp takes bins of the block in turn: its lanes filter the collected entries for those that cover the
//      bin, 32 at a time each lane stages its own item IN REGISTERS (same layout as the ring's items; only the rare slow
//      path gets a copy on the thread's stack) and evaluates the same fast / slow term functions, a fixed butterfly adds
//      the lanes, and lane 0 adds the round's sum to the bin's accumulator.
// Every bin is written once, with no atomics and no list in global memory, in an order that depends on the data only.
// This is the paper's own map -- the segment of every (f, voice) predetermined (L105) -- with the threads over the
// voices of a frequency instead of over the frequencies of a voice.  The Eq. 12 inner products are formed from the
// block's accumulators (one range per block for k_inner_reduce).
// ---------------------------------------------------------------------------------------------------------
#define FDEMRI_BIN_WARPS 8
#define FDEMRI_BQ1 256               // per warp: voice-signs waiting for level 2 (>= 31 + 32 * L1U, L1U = 4)
#define FDEMRI_BQ2 512               // per warp: rows waiting for level 3
#define FDEMRI_BREG 256              // per warp: entries collected per round

struct FdemriBinWarpQ {
    unsigned q1[FDEMRI_BQ1];
    unsigned q2[FDEMRI_BQ2];
    uint2 reg[FDEMRI_BREG];          // {key, first bin | last bin << 8, both relative to the block}
};
struct FdemriBinSmem {
    double4 acc[FDEMRI_BIN_BLOCK];
    FdemriBinWarpQ wq[FDEMRI_BIN_WARPS];
    unsigned short wlist[FDEMRI_BIN_WARPS][64];
    int reg_cnt[FDEMRI_BIN_WARPS];
    int cur_block;
};
struct FdemriBinEmit {
    uint2* reg;
    int n, Sp, b0, b1;
    __device__ __forceinline__ int room() const { return FDEMRI_BREG - n; }
    __device__ __forceinline__ void store(int off, int vsbr, int seg, int lo, int hi) {
        reg[n + off] = make_uint2((unsigned)(vsbr * Sp + seg), (unsigned)(max(lo, b0) - b0) | ((unsigned)(min(hi, b1) - b0) << 8));
    }
    __device__ __forceinline__ void advance(int k) { n += k; }
};

__global__ void __launch_bounds__(FDEMRI_BIN_WARPS * 32, 2) k_bin_sum(SumArgs a) {
    extern __shared__ __align__(16) unsigned char fdemri_bin_smem[];
    FdemriBinSmem* sm = reinterpret_cast<FdemriBinSmem*>(fdemri_bin_smem);
    const FdemriDims& d = a.d;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const unsigned full = 0xffffffffu, lt = (1u << lane) - 1u;
    const int V = d.n_modes, S = d.n_seg, Sp = 32 * d.n_groups, NB = d.tile_bins;     // NB <= FDEMRI_BIN_BLOCK
    const int part = ((2 * V + FDEMRI_BIN_WARPS - 1) / FDEMRI_BIN_WARPS + 31) & ~31;     // voice-signs per warp
    unsigned n_airy = 0, n_slow = 0, errs = 0;
    unsigned long long n_acc = 0;
    for (;;) {
        __syncthreads();                                             // the previous block's accumulators have been read
        if (tid == 0) sm->cur_block = (int)atomicAdd(a.tile_counter, 1u);
        if (tid < FDEMRI_BIN_BLOCK) sm->acc[tid] = make_double4(0.0, 0.0, 0.0, 0.0);
        __syncthreads();
        if (sm->cur_block >= a.total_tiles) break;
        // A CTA gets only a few blocks (config 3: 1250 for 296 CTAs), so the blocks handed out last decide how long the
        // last CTA runs alone.  The blocks of an item go out from the TOP of the grid down: the expensive terms -- the
        // slow path near the extrema of F and at small |X|, where the inspiral ends -- sit at the
        // highest frequencies a voice reaches, so the tail is made of the cheap blocks (config 3: 0.273 -> 0.251 ms;
        // sorting the blocks by the number of voice bands that cover them was measured too: 0.260 ms plus 27 us of sort).
        const int b = sm->cur_block / d.n_tiles, blk = d.n_tiles - 1 - (sm->cur_block - b * d.n_tiles);
        const int gb = b * d.n_tiles + blk;
        const int i0 = blk * NB;
        const int i1 = (int)min((int64_t)i0 + NB - 1, d.n_freq - 1);
        const int wbase = (a.n_angles > 1 ? b : 0) * V;
        const size_t rbase = (size_t)b * V * S;
        const bool in_band = i0 <= __ldg(a.iband + 2 * b + 1) - 1 && i1 >= 0x7fffffff - __ldg(a.iband + 2 * b);
        FdemriScan sc;
        const int vs0 = min(wid * part, 2 * V), vs1 = min(vs0 + part, 2 * V);
        fdemri_scan_init<FDEMRI_BQ2>(sc, a, b, vs0, in_band ? vs1 : vs0, i0, i1);
        FdemriBinWarpQ* wq = &sm->wq[wid];
        int more;
        do {
            // ---- A: this warp's part of the voice range: entries that meet the block, as many as fit ----
            FdemriBinEmit em;
            em.reg = wq->reg; em.n = 0; em.Sp = Sp; em.b0 = i0; em.b1 = i1;
            int rc;
            while ((rc = fdemri_scan_step<FDEMRI_BQ1, FDEMRI_BQ2, 4>(sc, wq->q1, wq->q2, lane, em)) == 1) {}
            if (lane == 0) sm->reg_cnt[wid] = em.n;
            more = __syncthreads_or(rc != 0);
            // ---- B: bins of the block, a warp each ----
            for (int t = wid; i0 + t <= i1; t += FDEMRI_BIN_WARPS) {
                const double f = fdemri_freq(d, i0 + t);
                double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
                unsigned wl_head = 0u, wl_tail = 0u;
                bool any = false;
                // evaluates the first `nl` waiting entries, a lane each
                auto evaluate = [&](int nl) {
                    if (lane < nl) {
                        const unsigned idx = sm->wlist[wid][(wl_head + (unsigned)lane) & 63u];
                        const unsigned key = sm->wq[idx / FDEMRI_BREG].reg[idx % FDEMRI_BREG].x;
                        const int vsbr = (int)(key / (unsigned)Sp), seg = (int)(key - (unsigned)vsbr * (unsigned)Sp);
                        const int vs = vsbr / 3, br = vsbr - 3 * vs;
                        const int v = vs >> 1;
                        // the lane's item stays in registers (every index below is a constant after inlining); only the
                        // rare slow path gets a copy on the thread's stack, which its out-of-line function reads
                        __align__(16) double item[S_DOUBLES];
                        fdemri_stage_item(item, a.rec + (rbase + (size_t)v * S + seg) * R_DOUBLES, a.wts[wbase + v], 0, 0,
                                          (unsigned)(vs & 1), (unsigned)br);
                        const unsigned flags = (unsigned)(*reinterpret_cast<const int2*>(item)).y;
                        const double sf = fdemri_xorsign(f, (flags & 4u) << 29);
                        double Tr = 0.0, Ti = 0.0;
                        bool ok = false;
                        if (!(flags & 1u)) ok = fdemri_term_fast(item, sf, Tr, Ti);
                        if (!ok) {
                            __align__(16) double it[S_DOUBLES];          // a copy on the thread's stack (local memory)
#pragma unroll
                            for (int q = 0; q < S_DOUBLES; ++q) it[q] = item[q];
                            const FdemriSlowOut o = fdemri_term_slow(it, sf, flags);
                            Tr = o.tre; Ti = o.tim;
                            n_airy += o.info & 1u; n_slow += (o.info >> 1) & 1u; errs |= o.info >> 4;
                        }
                        a0 = fma(item[S_WP], Tr, a0); a1 = fma(item[S_SWP], Ti, a1); a2 = fma(item[S_NWX], Ti, a2); a3 = fma(item[S_SWX], Tr, a3);
                        ++n_acc;
                    }
                    wl_head += (unsigned)nl;
                    any = true;
                };
                for (int r = 0; r < FDEMRI_BIN_WARPS; ++r) {
                    const int cnt = sm->reg_cnt[r];
                    for (int j0 = 0; j0 < cnt; j0 += 32) {
                        const int j = j0 + lane;
                        bool hit = false;
                        if (j < cnt) {
                            const unsigned span = sm->wq[r].reg[j].y;
                            hit = t >= (int)(span & 255u) && t <= (int)(span >> 8);
                        }
                        const unsigned mk = __ballot_sync(full, hit);
                        if (hit) sm->wlist[wid][(wl_tail + (unsigned)__popc(mk & lt)) & 63u] = (unsigned short)(r * FDEMRI_BREG + j);
                        wl_tail += (unsigned)__popc(mk);
                        __syncwarp();
                        if (wl_tail - wl_head >= 32u) evaluate(32);
                    }
                }
                if (wl_tail != wl_head) evaluate((int)(wl_tail - wl_head));
                if (any) {                                           // (warp-uniform)
#pragma unroll
                    for (int o = 16; o; o >>= 1) {
                        a0 += __shfl_xor_sync(full, a0, o); a1 += __shfl_xor_sync(full, a1, o);
                        a2 += __shfl_xor_sync(full, a2, o); a3 += __shfl_xor_sync(full, a3, o);
                    }
                    if (lane == 0) {
                        double4 s4 = sm->acc[t];
                        s4.x += a0; s4.y += a1; s4.z += a2; s4.w += a3;
                        sm->acc[t] = s4;
                    }
                }
            }
            __syncthreads();                                         // the collected entries may be overwritten
        } while (more);
        // ---- outputs of the block: the waveform (S4) and / or its share of the inner products of Eq. 12 ----
        if (wid == 0) {
            const int64_t bin = (int64_t)i0 + lane;
            const bool valid = lane < NB && bin <= i1;
            const double4 h = sm->acc[lane];                          // (zero past the block and past the grid)
            if (a.hp && valid) {
                const size_t o = ((size_t)b * d.n_freq + bin) * 2;
                *reinterpret_cast<double2*>(a.hp + o) = make_double2(h.x, h.y);
                *reinterpret_cast<double2*>(a.hx + o) = make_double2(h.z, h.w);
            }
            if (a.inner_part) {
                double4 u = h;
                bool use = valid;
                if (a.inner_edge) {
                    // Hann window as the 3-point filter h_k/2 - h_{k-1}/4 - h_{k+1}/4 (L145): the first and the last bin
                    // of the block need a bin of a neighbouring block and are left to k_inner_reduce
                    if (lane < 2 || (lane >= NB - 2 && lane < NB))
                        *reinterpret_cast<double4*>(a.inner_edge + ((size_t)gb * 4 + (lane < 2 ? lane : lane - (NB - 4))) * 4) = h;
                    double4 l, r;
                    l.x = __shfl_up_sync(full, h.x, 1); l.y = __shfl_up_sync(full, h.y, 1);
                    l.z = __shfl_up_sync(full, h.z, 1); l.w = __shfl_up_sync(full, h.w, 1);
                    r.x = __shfl_down_sync(full, h.x, 1); r.y = __shfl_down_sync(full, h.y, 1);
                    r.z = __shfl_down_sync(full, h.z, 1); r.w = __shfl_down_sync(full, h.w, 1);
                    u = fdemri_hann3(l, h, r);
                    use = valid && lane != 0 && lane != NB - 1;
                }
                double hh = 0.0, dr = 0.0, di = 0.0;
                if (use) fdemri_inner_bin(u, bin, a.weight, a.dplus, a.dcross, hh, dr, di);
#pragma unroll
                for (int o = 16; o; o >>= 1) {
                    hh += __shfl_xor_sync(full, hh, o);
                    dr += __shfl_xor_sync(full, dr, o);
                    di += __shfl_xor_sync(full, di, o);
                }
                if (lane == 0) *reinterpret_cast<double4*>(a.inner_part + (size_t)gb * 4) = make_double4(hh, dr, di, 0.0);
            }
        }
    }
    for (int o = 16; o; o >>= 1) {
        n_airy += __shfl_xor_sync(full, n_airy, o);
        n_slow += __shfl_xor_sync(full, n_slow, o);
        errs |= __shfl_xor_sync(full, errs, o);
        n_acc += __shfl_xor_sync(full, n_acc, o);
    }
    if (lane == 0) {
        if (n_airy) atomicAdd(a.stats + 4, (unsigned long long)n_airy);
        if (n_slow) atomicAdd(a.stats + 7, (unsigned long long)n_slow);
        if (errs) atomicOr(a.stats + 9, (unsigned long long)errs);
        if (n_acc) atomicAdd(a.stats + 8, n_acc);                  // accumulated terms (= n_evals of the map, P9)
    }
}
