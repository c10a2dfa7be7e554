// fdemri_sum.cuh -- S3 + S4: the output-tiled harmonic sum (the hot loop).
//
// Each CTA owns a tile of FDEMRI_TILE consecutive bins of one batch item (one bin per thread, accumulators in
// registers), walks the item's strips in their fixed (voice, sign, time) order, and for every strip that
// covers its bin evaluates the term of Eq. 9:
//     A(t) g(X)/sqrt|Fdot| exp{i[2 pi s f t - Phi(t)]},   t = t_k + tau,  F(tau) = s f  (Eq. 6)
// and adds it with the harmonic weights (Eq. 1).  Every bin is written once (S4): no atomics, and the
// summation order of a bin never depends on scheduling, so results are bitwise reproducible.
// The paper's own layout -- one block per (voice, segment), atomicAdd into global memory (L121) -- is prior art.
#pragma once
#include "fdemri_common.cuh"
#include "airy_tables.inc"

struct SumArgs {
    FdemriDims d;
    const double* rec;        // [B][V][S][R_DOUBLES]
    const int2* ent;          // [B][V][2][ent_max]
    const int4* dense;        // [B][dense_cap]
    const int* n_dense;       // [B]
    int dense_cap;
    const double4* wts;       // [n_angles][V]
    int n_angles;
    double* hp;               // [B][n_freq][2]
    double* hx;
    unsigned int* tile_counter;
    unsigned long long* stats;
    int total_tiles;
};

// asymptotic series of g(X) e^{+i pi/4 sgn X} = sum_k i^k a_k u^k, u = 1/X, a_k = prod_j (4/9-(2j-1)^2)/(k! 8^k)
__device__ __forceinline__ void fdemri_g_series(double u, double& re, double& im) {
    double u2 = u * u;
    if (fabs(u) <= 2.5e-3) {          // |X| >= 400: through a_4, error < 1.2e-14
        re = fma(u2, fma(u2, 0.05764919041266972, -0.037133487654320986), 1.0);
        im = u * fma(u2, 0.03799305912780064, -0.06944444444444445);
    } else {                          // 28 <= |X| < 400: through a_12, error < 2e-15
        double r = 1533.1694320127956;
        r = fma(r, u2, -55.62278536591708);
        r = fma(r, u2, 3.079453030173167);
        r = fma(r, u2, -0.2915913992307505);
        r = fma(r, u2, 0.05764919041266972);
        r = fma(r, u2, -0.037133487654320986);
        re = fma(r, u2, 1.0);
        double q = 278.46508077760257;
        q = fma(q, u2, -12.341573332345238);
        q = fma(q, u2, 0.8776669695100169);
        q = fma(q, u2, -0.11609906402551541);
        q = fma(q, u2, 0.03799305912780064);
        q = fma(q, u2, -0.06944444444444445);
        im = q * u;
    }
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

// One term.  R: the (voice, segment) record; sgn = +-1; f the bin frequency; brB: second branch of a turnover
// segment; w = {w+, wx, m phi/2pi}.  Accumulates into acc[4] = {Re h+, Im h+, Re hx, Im hx}.
__device__ __forceinline__ void fdemri_term(const double* __restrict__ R, double sgn, double f, int brB,
                                            const double4 w, double acc[4], unsigned int& n_airy,
                                            unsigned int& bad) {
    const double FA = R[R_FA], FB = R[R_FB], FC = R[R_FC], FD = R[R_FD];
    const double h = R[R_H];
    const double sf = sgn * f;
    double tau, Fd;
    if (R[R_TYPE] == 0.0) {
        // monotone segment: seed from the stored inverse cubic, then Newton on F(tau) - s f
        const double x = sf - FA;
        tau = x * fma(x, fma(x, R[R_Q3], R[R_Q2]), R[R_Q1]);
        tau = fmin(fmax(tau, 0.0), h);
        const double tol = 1e-14 * h;
        int it = 0;
        for (; it < 40; ++it) {
            double G = fma(tau, fma(tau, fma(tau, FD, FC), FB), -x);
            double dG = fma(tau, fma(tau, 3.0 * FD, 2.0 * FC), FB);
            double delta = G / dG;
            tau = fmin(fmax(tau - delta, 0.0), h);      // the root is inside [0, h] (membership, R6)
            if (fabs(delta) <= tol) break;
        }
        if (it == 40) bad |= 8u;
        Fd = fma(tau, fma(tau, 3.0 * FD, 2.0 * FC), FB);
    } else {
        // turnover segment: F(tau) - F_e = z^2 (c2 + FD z), z = tau - tau_e; branch A: z < 0, branch B: z > 0
        const double te = R[R_Q1], Fe = R[R_Q2], c2 = R[R_Q3];
        const double Delta = sf - Fe;
        double ratio = Delta / c2;
        double z = sqrt(fmax(ratio, 0.0));
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
        if (it == 40) bad |= 8u;
        z = brB ? fmin(fmax(z, 0.0), h - te) : fmax(fmin(z, 0.0), -te);
        tau = te + z;
        Fd = z * fma(3.0 * FD, z, 2.0 * c2);          // exact factorisation, no cancellation near Fdot = 0
    }
    const double Fdd = fma(6.0 * FD, tau, 2.0 * FC);
    if (Fd == 0.0 && Fdd == 0.0) return;               // R10: no term
    // amplitude (two cubics)
    const double Are = fma(tau, fma(tau, fma(tau, R[R_AR + 3], R[R_AR + 2]), R[R_AR + 1]), R[R_AR]);
    const double Aim = fma(tau, fma(tau, fma(tau, R[R_AI + 3], R[R_AI + 2]), R[R_AI + 1]), R[R_AI]);
    // phase in cycles (R9): (s f) t_k exactly as p + e, local cubic in tau, knot phase from the record
    const double tk = R[R_TK];
    const double p = __dmul_rn(sf, tk);
    const double e = __fma_rn(sf, tk, -p);
    const double pr = p - rint(p);
    double wv = (sf - R[R_BH]) - R[R_BL];
    const double loc = tau * fma(tau, fma(tau, R[R_ND], R[R_NC]), wv);
    double cyc = ((pr + e) + (R[R_PC] + w.z)) + loc;
    // g(X)/sqrt|Fdot|
    const double aFd = fabs(Fd);
    const double sig = (Fd >= 0.0) ? 1.0 : -1.0;
    double Sre, Sim;
    if (6.283185307179586 * aFd * aFd * aFd >= 84.0 * Fdd * Fdd) {
        // |X| >= 28: asymptotic series; the e^{-+ i pi/4} goes into the phase
        const double y = rsqrt(aFd);
        const double y2 = y * y;
        const double pq = Fdd * y2;
        const double u = 0.477464829275686 * pq * pq * y2 * sig;    // 1/X = 3 Fdd^2 / (2 pi Fd^3)
        double gr, gi;
        fdemri_g_series(u, gr, gi);
        Sre = gr * y;
        Sim = gi * y;
        cyc -= 0.125 * sig;
    } else {
        // |X| < 28: regular Airy form  e^{-iX} pi kap [Ai(-yy) -+ i Bi(-yy)],  kap = (pi|Fddot|)^(-1/3)
        const double kap = rcbrt(3.141592653589793 * fabs(Fdd));
        const double k2 = kap * kap;
        const double yy = k2 * k2 * 9.869604401089358 * Fd * Fd;
        double ai, bi;
        fdemri_airy_neg(yy, ai, bi);
        const double X = 0.6666666666666666 * sig * yy * sqrt(yy);
        cyc -= X * 0.15915494309189535;
        Sre = 3.141592653589793 * kap * ai;
        Sim = -sig * 3.141592653589793 * kap * bi;
        ++n_airy;
    }
    double sn, cs;
    sincospi(2.0 * cyc, &sn, &cs);
    const double Ere = Sre * cs - Sim * sn, Eim = Sre * sn + Sim * cs;
    const double Tre = Are * Ere - Aim * Eim, Tim = Are * Eim + Aim * Ere;
    // weights (O2): s=+1: h+ += w+ T, hx += i wx T;  s=-1: h+ += w+ conj(T), hx += conj(i wx T)
    acc[0] = fma(w.x, Tre, acc[0]);
    acc[1] = fma(sgn * w.x, Tim, acc[1]);
    acc[2] = fma(-w.y, Tim, acc[2]);
    acc[3] = fma(sgn * w.y, Tre, acc[3]);
}

__global__ void __launch_bounds__(FDEMRI_TILE) k_tile_sum(SumArgs a) {
    __shared__ int s_tile;
    __shared__ int4 s_list[FDEMRI_TILE];     // {strip lo, strip hi, (vs<<1)|dir, e_first | e_last<<16} (absolute entries)
    __shared__ int s_warp_cnt[FDEMRI_TILE / 32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const FdemriDims& d = a.d;
    const int V = d.n_modes;
    unsigned int n_airy = 0, bad = 0;
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
        const int nd = a.n_dense[b];
        const int4* dense_b = a.dense + (size_t)b * a.dense_cap;
        const double4* wts_b = a.wts + (size_t)(a.n_angles > 1 ? b : 0) * V;
        for (int base = 0; base < nd; base += FDEMRI_TILE) {
            // ---- candidate strips of this chunk, kept in order (deterministic compaction) ----
            const int c = base + tid;
            bool hit = false;
            int4 item = make_int4(0, 0, 0, 0);
            if (c < nd) {
                int4 s = dense_b[c];
                if (s.x <= tile_hi && s.y >= tile_lo) {
                    hit = true;
                    const int vs = s.z >> 1, dir = s.z & 1;
                    const int e0 = s.w & 0xffff, ne = s.w >> 16;
                    const int2* E = a.ent + ((size_t)b * 2 * V + vs) * d.ent_max + e0;
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
                    item = make_int4(s.x, s.y, s.z, (e0 + ea) | ((e0 + eb) << 16));
                }
            }
            const unsigned ballot = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) s_warp_cnt[wid] = __popc(ballot);
            __syncthreads();
            int off = 0, cnt = 0;
#pragma unroll
            for (int i = 0; i < FDEMRI_TILE / 32; ++i) {
                int ci = s_warp_cnt[i];
                if (i < wid) off += ci;
                cnt += ci;
            }
            if (hit) s_list[off + __popc(ballot & ((1u << lane) - 1u))] = item;
            __syncthreads();
            // ---- evaluate ----
            if (valid) {
                for (int j = 0; j < cnt; ++j) {
                    const int4 s = s_list[j];
                    if (bin < s.x || bin > s.y) continue;
                    const int vs = s.z >> 1, dir = s.z & 1;
                    const int v = vs >> 1;
                    const double sgn = (vs & 1) ? -1.0 : 1.0;
                    const int2* E = a.ent + ((size_t)b * 2 * V + vs) * d.ent_max;
                    int e = s.w & 0xffff;
                    const int eb = s.w >> 16;
                    const int ibin = (int)bin;
                    if (dir) { while (e < eb && E[e + 1].x <= ibin) ++e; }
                    else { while (e < eb && E[e].x > ibin) ++e; }
                    const int segf = E[e].y;
                    const int seg = segf & 0x3fffffff;
                    const double* R = a.rec + (((size_t)b * V + v) * d.n_seg + seg) * R_DOUBLES;
                    fdemri_term(R, sgn, f, (segf >> 30) & 1, wts_b[v], acc, n_airy, bad);
                }
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
        n_airy += __shfl_xor_sync(0xffffffffu, n_airy, o);
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if (lane == 0) {
        if (n_airy) atomicAdd(a.stats + 4, (unsigned long long)n_airy);
        if (bad) atomicOr(a.stats + 5, (unsigned long long)bad);
    }
}
