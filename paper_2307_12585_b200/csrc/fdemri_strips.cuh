// fdemri_strips.cuh -- S2b: bin intervals of every (voice, sign, segment-branch) and the strips they form.
//
// Membership (R6-R8), decided on doubles only: the knot values F_k (fdemri_knotF), the extremum
// value F_e of a turnover segment (record slot R_Q2) and the bin frequencies f_i.
//   branch from value Va (start, in time) to Vb (end):
//     normal segment        : Va = F_k included, Vb = F_{k+1} excluded          (half-open in time, R6)
//     turnover, 1st branch  : Va = F_k included, Vb = F_e included               (R7)
//     turnover, 2nd branch  : Va = F_e excluded, Vb = F_{k+1} excluded
//   a bin f_i > 0 belongs to the branch for sign s when s*f_i lies between Va and Vb under those rules.
#pragma once
#include "fdemri_common.cuh"

// first bin index with f_i >= x  (n_freq if none)
__device__ int64_t fdemri_first_ge(const FdemriDims& d, double x) {
    int64_t n = d.n_freq;
    if (d.freq) {
        int64_t lo = 0, hi = n;
        while (lo < hi) { int64_t mid = (lo + hi) >> 1; if (__ldg(d.freq + mid) < x) lo = mid + 1; else hi = mid; }
        return lo;
    }
    double g = ceil((x - d.f0) / d.df);
    int64_t i = (g <= 0.0) ? 0 : (g >= (double)n ? n : (int64_t)g);
    while (i > 0 && fdemri_freq(d, i - 1) >= x) --i;
    while (i < n && fdemri_freq(d, i) < x) ++i;
    return i;
}
// first bin index with f_i > x
__device__ int64_t fdemri_first_gt(const FdemriDims& d, double x) {
    int64_t n = d.n_freq;
    if (d.freq) {
        int64_t lo = 0, hi = n;
        while (lo < hi) { int64_t mid = (lo + hi) >> 1; if (__ldg(d.freq + mid) <= x) lo = mid + 1; else hi = mid; }
        return lo;
    }
    double g = floor((x - d.f0) / d.df) + 1.0;
    int64_t i = (g <= 0.0) ? 0 : (g >= (double)n ? n : (int64_t)g);
    while (i > 0 && fdemri_freq(d, i - 1) > x) --i;
    while (i < n && fdemri_freq(d, i) <= x) ++i;
    return i;
}

struct StripRaw {   // per (item, voice, sign), FDEMRI_MAX_STRIPS of them
    int lo, hi;     // inclusive bin range
    int e0;         // first entry (index into this (voice, sign)'s entry list)
    int n_dir;      // (number of entries << 1) | (1 if bins increase with time)
};

// One thread per (batch item, voice, sign).  ent: [B][V][2][ent_max] int4 {first bin, last bin, seg | branchB<<30, 0}
// of every non-empty (segment, branch), in time order;  n_ent: [B][V][2] their number
__global__ void k_strips(FdemriDims d, const int* __restrict__ lmn, const double* __restrict__ f_phi,
                         const double* __restrict__ f_r, const double* __restrict__ rec, int4* __restrict__ ent,
                         int* __restrict__ n_ent, StripRaw* __restrict__ strips, int* __restrict__ n_strips,
                         unsigned long long* __restrict__ stats) {
    size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t total = (size_t)d.n_batch * d.n_modes * 2;
    if (id >= total) return;
    int sg = (int)(id & 1);                     // 0: s = +1, 1: s = -1
    size_t bv = id >> 1;
    int v = (int)(bv % d.n_modes);
    int b = (int)(bv / d.n_modes);
    int m = lmn[3 * v + 1], n = lmn[3 * v + 2];
    const double s = sg ? -1.0 : 1.0;
    const double* R = rec + bv * (size_t)d.n_seg * R_DOUBLES;
    int4* E = ent + id * (size_t)d.ent_max;
    StripRaw* ST = strips + id * FDEMRI_MAX_STRIPS;
    const int64_t first_pos = fdemri_first_gt(d, 0.0);      // bins with f > 0 only (R13)
    int ne = 0, ns = 0;
    unsigned long long evals = 0, flags = 0;
    // open strip state
    bool open = false; int cur_dir = 0; int64_t cur_lo = 0, cur_hi = 0; int cur_e0 = 0, cur_n = 0;
    const double Flast = fdemri_knotF(m, n, f_phi[(size_t)b * d.n_knots + d.n_knots - 1],
                                      f_r[(size_t)b * d.n_knots + d.n_knots - 1]);
    for (int k = 0; k < d.n_seg; ++k) {
        const double* Rk = R + (size_t)k * R_DOUBLES;
        double Fk = Rk[R_FA];
        double Fk1 = (k + 1 < d.n_seg) ? Rk[R_DOUBLES + R_FA] : Flast;
        int type = (int)Rk[R_TYPE];
        if (type == 2) continue;
        int nbr = (type == 1) ? 2 : 1;
        for (int br = 0; br < nbr; ++br) {
            double Va, Vb; bool a_incl, b_incl;
            if (type == 0) { Va = Fk; Vb = Fk1; a_incl = true; b_incl = false; }
            else if (br == 0) { Va = Fk; Vb = Rk[R_Q2]; a_incl = true; b_incl = true; }
            else { Va = Rk[R_Q2]; Vb = Fk1; a_incl = false; b_incl = false; }
            if (Va == Vb) continue;
            double lo_v = fmin(Va, Vb), hi_v = fmax(Va, Vb);
            bool lo_incl = (Va < Vb) ? a_incl : b_incl;
            bool hi_incl = (Va < Vb) ? b_incl : a_incl;
            double flo = sg ? -hi_v : lo_v, fhi = sg ? -lo_v : hi_v;
            bool flo_incl = sg ? hi_incl : lo_incl, fhi_incl = sg ? lo_incl : hi_incl;
            if (!(fhi > 0.0)) continue;
            int64_t lo = flo_incl ? fdemri_first_ge(d, flo) : fdemri_first_gt(d, flo);
            int64_t hi1 = fhi_incl ? fdemri_first_gt(d, fhi) : fdemri_first_ge(d, fhi);
            if (lo < first_pos) lo = first_pos;
            if (lo >= hi1) continue;
            int dir = (s * (Vb - Va) > 0.0) ? 1 : 0;          // bins increase with time?
            bool adjacent = open && dir == cur_dir && (dir ? (lo == cur_hi + 1) : (hi1 == cur_lo));
            if (!adjacent) {
                if (open) {
                    if (ns < FDEMRI_MAX_STRIPS) ST[ns++] = StripRaw{(int)cur_lo, (int)cur_hi, cur_e0, (cur_n << 1) | cur_dir};
                    else flags |= 2ull;
                }
                open = true; cur_dir = dir; cur_lo = lo; cur_hi = hi1 - 1; cur_e0 = ne; cur_n = 0;
            } else {
                if (dir) cur_hi = hi1 - 1; else cur_lo = lo;
            }
            if (ne < d.ent_max) {
                E[ne++] = make_int4((int)lo, (int)(hi1 - 1), k | (br << 30), 0);
                ++cur_n;
                evals += (unsigned long long)(hi1 - lo);
            } else {
                flags |= 2ull;
            }
        }
    }
    if (open) {
        if (ns < FDEMRI_MAX_STRIPS) ST[ns++] = StripRaw{(int)cur_lo, (int)cur_hi, cur_e0, (cur_n << 1) | cur_dir};
        else flags |= 2ull;
    }
    n_strips[id] = ns;
    n_ent[id] = ne;
    if (ne) atomicAdd(stats + 0, (unsigned long long)ne);
    if (ns) atomicAdd(stats + 1, (unsigned long long)ns);
    if (evals) atomicAdd(stats + 2, evals);
    if (flags) atomicOr(stats + 5, flags);
}

// Dense per-item strip list in (voice, sign, time) order: one CTA per batch item.
// dense: [B][cap] int4 {lo, hi, (vs << 1) | dir, e0 | (n << 16)};  n_dense: [B]
__global__ void k_strip_compact(int V, int cap, const StripRaw* __restrict__ strips, const int* __restrict__ n_strips,
                                int4* __restrict__ dense, int* __restrict__ n_dense, int2* __restrict__ bin_range) {
    __shared__ int s_scan[1024];
    __shared__ int s_base;
    __shared__ int s_min, s_max;
    if (threadIdx.x == 0) { s_min = 0x7fffffff; s_max = -1; }
    int my_min = 0x7fffffff, my_max = -1;
    int b = blockIdx.x;
    int nvs = 2 * V;
    if (threadIdx.x == 0) s_base = 0;
    __syncthreads();
    for (int start = 0; start < nvs; start += blockDim.x) {
        int vs = start + threadIdx.x;
        int cnt = (vs < nvs) ? n_strips[(size_t)b * nvs + vs] : 0;
        s_scan[threadIdx.x] = cnt;
        __syncthreads();
        for (int off = 1; off < blockDim.x; off <<= 1) {          // inclusive Hillis-Steele scan
            int add = (threadIdx.x >= off) ? s_scan[threadIdx.x - off] : 0;
            __syncthreads();
            s_scan[threadIdx.x] += add;
            __syncthreads();
        }
        int pos = s_base + s_scan[threadIdx.x] - cnt;
        if (vs < nvs) {
            const StripRaw* ST = strips + ((size_t)b * nvs + vs) * FDEMRI_MAX_STRIPS;
            for (int j = 0; j < cnt; ++j) {
                StripRaw r = ST[j];
                my_min = min(my_min, r.lo);
                my_max = max(my_max, r.hi);
                if (pos + j < cap)
                    dense[(size_t)b * cap + pos + j] = make_int4(r.lo, r.hi, (vs << 1) | (r.n_dir & 1), r.e0 | ((r.n_dir >> 1) << 16));
            }
        }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) s_base += s_scan[threadIdx.x];
        __syncthreads();
    }
    atomicMin(&s_min, my_min);
    atomicMax(&s_max, my_max);
    __syncthreads();
    if (threadIdx.x == 0) {
        n_dense[b] = min(s_base, cap);
        bin_range[b] = make_int2(s_min, s_max);
    }
}
