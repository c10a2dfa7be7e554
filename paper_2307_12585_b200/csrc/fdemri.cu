// fdemri.cu -- host side of libfdemri (C ABI of include/fdemri.h).  One translation unit: the kernels live
// in the .cuh files included below.  Build: see paper_2307_12585_b200/build.py
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo -Xcompiler -fPIC -shared
#include "../../include/fdemri.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <cstring>
#include <mutex>
#include <new>
#include <unordered_map>
#include <vector>

#include "fdemri_common.cuh"
#include "fdemri_map.cuh"
#include "fdemri_splines.cuh"
#include "fdemri_select.cuh"
#include "fdemri_sum.cuh"
#include "fdemri_td.cuh"

struct fdemri_plan_s {
    FdemriDims d;
    std::vector<int32_t> lmn;
    std::vector<int32_t> kk;       // polar harmonic k per voice (general voices, fdemri_plan_kerr); empty otherwise
    int* k_dev;                    // NULL unless kk is in use
    double *sh2_hi, *sh2_lo;       // splines of (f_theta, Phi_theta), same layout as sh_hi/sh_lo; NULL unless kk
    const double* t_knots_dev;
    // work space carve-up (device pointers)
    void* ws;
    size_t ws_bytes;
    int* lmn_dev;
    int* lm_index_dev;             // [V] index of the voice's (l, m) in the weight table
    int4* wmeta_dev;               // [n_lm][2] {terms, p0, q0, offset} for +m and -m
    double* wcoef_dev;             // Wigner-sum coefficients
    std::vector<int> lm_index;
    std::vector<int4> wmeta;
    std::vector<double> wcoef;
    double *sh_hi, *sh_lo, *rec;
    int2* ent;                     // [B][V][2][3][S] bin intervals of the segment branches
    int4* gband;                   // [B][V][2][G] bands of the groups of 32 segments
    int2* vband;                   // [B][V][2] bands of the voice-signs
    int* iband;                    // [B][2] {0x7fffffff - lo, hi + 1} of the item ({0, 0}: empty)
    unsigned long long* item_evals;// [B] mode-bin evaluations of the map, per batch item
    size_t build_clear_bytes;      // stats .. item_evals, cleared by one memset per build
    double* inner_part;            // [ranges][4] partial inner products (a range: 64 bins of a consumer warp, or a block)
    double* inner_edge;            // [ranges][4][4] edge bins for the Hann filter
    double* sel_total;             // [B][n_knots] total power per time step (mode selection)
    const unsigned char* mode_mask;// [B][V] borrowed from the caller, or NULL: every mode is summed
    double4* wts;
    double* angles;
    unsigned long long* stats;     // [0..5], [7], [8] = fdemri_stats, [6] = tile counter (low 32 bits), [9] = flags of the
                                   // last sum; 16 slots
    double* angle_stage;           // pinned host buffer [2 * n_batch]: the angles of the last sum, read by its async copy
    bool built;
    cudaStream_t last_stream;
    int sm_count;
    int sum_blocks_per_sm;         // resident CTAs of k_tile_sum per SM (0: not queried yet)
    uint32_t flags;
    cudaEvent_t ev0, ev1;
    cudaStream_t side;             // the amplitude splines run beside the shared ones (fork/join on two events)
    cudaEvent_t ev_fork, ev_join;
    bool lut_built;                // explicit grids: the bucket table of the frequency array has been enqueued
    bool ev_valid;
    cudaEvent_t ev_angles;         // the copy of the angles out of the pinned staging buffer has run
    bool last_stream_valid;
};

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// walks the carve-up; with base == nullptr only sizes are computed
static size_t carve(fdemri_plan_s* p, char* base) {
    const FdemriDims& d = p->d;
    size_t off = 0;
    const size_t B = d.n_batch, V = d.n_modes, S = d.n_seg;
    auto take = [&](size_t bytes) {
        char* ptr = base ? base + off : nullptr;
        off += align_up(bytes);
        return ptr;
    };
    p->lmn_dev = (int*)take(V * 3 * sizeof(int));
    const bool polar = !p->kk.empty();
    p->k_dev = polar ? (int*)take(V * sizeof(int)) : nullptr;
    p->sh2_hi = polar ? (double*)take(B * 4 * S * 4 * sizeof(double)) : nullptr;
    p->sh2_lo = polar ? (double*)take(B * 4 * S * 4 * sizeof(double)) : nullptr;
    p->lm_index_dev = (int*)take(V * sizeof(int));
    p->wmeta_dev = (int4*)take(p->wmeta.size() * sizeof(int4));
    p->wcoef_dev = (double*)take(p->wcoef.size() * sizeof(double));
    p->sh_hi = (double*)take(B * 4 * S * 4 * sizeof(double));
    p->sh_lo = (double*)take(B * 4 * S * 4 * sizeof(double));
    p->rec = (double*)take(B * V * S * R_DOUBLES * sizeof(double));
    p->ent = (int2*)take(B * V * 2 * (size_t)d.ent_max * sizeof(int2));
    p->gband = (int4*)take(B * V * 2 * (size_t)d.n_groups * sizeof(int4));
    p->vband = (int2*)take(B * V * 2 * sizeof(int2));
    // cleared together by one memset at the head of every build: keep the three adjacent and in this order
    p->stats = (unsigned long long*)take(16 * sizeof(unsigned long long));
    p->iband = (int*)take(B * 2 * sizeof(int));
    p->item_evals = (unsigned long long*)take(B * sizeof(unsigned long long));
    p->build_clear_bytes = base ? (size_t)((char*)p->item_evals - (char*)p->stats) + B * sizeof(unsigned long long) : 0;
    const size_t NT = B * (size_t)d.n_tiles;
    p->wts = (double4*)take(B * V * sizeof(double4));
    p->angles = (double*)take(B * 2 * sizeof(double));
    p->sel_total = (double*)take(B * (size_t)d.n_knots * sizeof(double));
    p->d.lut = d.lut_n ? (const int*)take(((size_t)d.lut_n + 1 + FDEMRI_LUT_HDR) * sizeof(int)) : nullptr;
    // partial inner products: one range per consumer warp of a tile, or per block of the bin-major kernel
    const size_t NR = d.bin_major ? NT : NT * FDEMRI_CWARPS;
    p->inner_part = (double*)take(NR * 4 * sizeof(double));
    p->inner_edge = (double*)take(NR * 16 * sizeof(double));
    return off;
}

// S0 table: -2Y_lm(theta, 0) = sqrt((2l+1)/4pi) d^l_{m,2}(theta) with the Wigner small-d function
//   d^l_{mp,2} = sum_k (-1)^{mp-2+k} sqrt((l+mp)!(l-mp)!(l+2)!(l-2)!) / [(l+2-k)! k! (mp-2+k)! (l-mp-k)!]
//                      cos(theta/2)^{2l+2-mp-2k} sin(theta/2)^{mp-2+2k}
// Everything but the powers depends on (l, mp) only: tabulated once per distinct (l, m) for mp = +m and mp = -m
// (the latter with the (-1)^l of the partner voice folded in), in long double.
static void build_weight_table(fdemri_plan_s* p) {
    const int V = p->d.n_modes;
    p->lm_index.assign(V, 0);
    p->wmeta.clear();
    p->wcoef.clear();
    std::unordered_map<int, int> seen;           // l * 1024 + m -> table row
    for (int v = 0; v < V; ++v) {
        const int l = p->lmn[3 * v], m = p->lmn[3 * v + 1];
        const int code = l * 1024 + m;
        int row;
        const auto hit = seen.find(code);
        if (hit != seen.end()) {
            row = hit->second;
        } else {
            row = (int)seen.size();
            seen.emplace(code, row);
            const long double norm = sqrtl((2.0L * l + 1.0L) / (4.0L * 3.14159265358979323846264338327950288L));
            for (int which = 0; which < 2; ++which) {
                const int mp = which ? -m : m;
                const long double lpref = 0.5L * (lgammal(l + mp + 1.0L) + lgammal(l - mp + 1.0L) + lgammal(l + 3.0L) +
                                                  lgammal(l - 1.0L));
                const int k0 = std::max(0, 2 - mp), k1 = std::min(l + 2, l - mp);
                int4 meta;
                meta.x = std::max(0, k1 - k0 + 1);
                meta.y = 2 * l + 2 - mp - 2 * k0;
                meta.z = mp - 2 + 2 * k0;
                meta.w = (int)p->wcoef.size();
                for (int k = k0; k <= k1; ++k) {
                    const long double lt = lpref - lgammal(l + 2 - k + 1.0L) - lgammal(k + 1.0L) - lgammal(mp - 2 + k + 1.0L) -
                                           lgammal(l - mp - k + 1.0L);
                    long double c = norm * expl(lt);
                    if ((mp - 2 + k) & 1) c = -c;
                    if (which && (l & 1)) c = -c;
                    p->wcoef.push_back((double)c);
                }
                p->wmeta.push_back(meta);
            }
        }
        p->lm_index[v] = row;
    }
}

// frees whatever the plan owns (streams, events, the pinned angle buffer); also the error paths of plan_impl
static void release_plan(fdemri_plan_s* p) {
    if (!p) return;
    if (p->side) cudaStreamDestroy(p->side);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->ev0) cudaEventDestroy(p->ev0);
    if (p->ev1) cudaEventDestroy(p->ev1);
    if (p->ev_angles) cudaEventDestroy(p->ev_angles);
    if (p->angle_stage) cudaFreeHost(p->angle_stage);
    delete p;
}

static int plan_impl(fdemri_plan_t* out, int n_modes, const int32_t* lmn_host, const int32_t* k_host, int n_batch,
                     int n_knots, const double* t_knots_dev, int64_t n_freq, const double* freq_dev, double f0, double df,
                     uint32_t flags) {
    if (!out) return FDEMRI_ERR_INVALID_ARG;
    *out = nullptr;
    if (n_modes < 1 || n_modes > (1 << 20) || !lmn_host || n_batch < 1 || n_knots < 4 || n_knots > FDEMRI_MAX_KNOTS ||
        !t_knots_dev || n_freq < 1 || n_freq >= ((int64_t)1 << 31) - FDEMRI_TILE)
        return FDEMRI_ERR_INVALID_ARG;
    if (!freq_dev && !(df > 0.0 && std::isfinite(df) && std::isfinite(f0) && f0 >= 0.0)) return FDEMRI_ERR_INVALID_ARG;
    for (int v = 0; v < n_modes; ++v) {
        int l = lmn_host[3 * v], m = lmn_host[3 * v + 1], n = lmn_host[3 * v + 2];
        if (l < 2 || l > 60 || m < 0 || m > l || n < -100000 || n > 100000) return FDEMRI_ERR_INVALID_ARG;
        if (k_host && (k_host[v] < -100000 || k_host[v] > 100000)) return FDEMRI_ERR_INVALID_ARG;
    }
    /* Which sum kernel: tile-major when the entries are wide in bins (dense grids), bin-major
       when a bin interval holds only a few bins (sparse grids, section 3.3).  The entries of a voice split its
       band into n_seg pieces, so n_freq / n_seg bounds the bins per entry. */
    if ((flags & FDEMRI_FLAG_BIN_MAJOR) && (flags & FDEMRI_FLAG_TILE_MAJOR)) return FDEMRI_ERR_INVALID_ARG;
    const bool bin_major = (flags & FDEMRI_FLAG_BIN_MAJOR) ||
                           (!(flags & FDEMRI_FLAG_TILE_MAJOR) && n_freq < (int64_t)256 * (n_knots - 1));
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return FDEMRI_ERR_CUDA;
    /* bin-major: the largest block of bins (32, 16, 8) that still gives every resident CTA (two per SM) four blocks:
       a block costs a scan of all voice bands, so large blocks are cheap, but few blocks balance badly */
    int tile_bins = bin_major ? FDEMRI_BIN_BLOCK : FDEMRI_TILE;
#ifndef FDEMRI_BIN_BLOCKS_PER_SM
#define FDEMRI_BIN_BLOCKS_PER_SM 8
#endif
    while (bin_major && tile_bins > 8 &&
           (n_freq * (int64_t)n_batch) / tile_bins < (int64_t)FDEMRI_BIN_BLOCKS_PER_SM * prop.multiProcessorCount)
        tile_bins /= 2;
    int64_t n_tiles = (n_freq + tile_bins - 1) / tile_bins;
    if (n_tiles * (int64_t)n_batch >= ((int64_t)1 << 31)) return FDEMRI_ERR_INVALID_ARG;
    if ((int64_t)n_batch * n_modes * (n_knots - 1) >= ((int64_t)1 << 31)) return FDEMRI_ERR_INVALID_ARG;   /* 32-bit record index */
    if ((int64_t)n_modes * 6 * (n_knots + 31) >= ((int64_t)1 << 27)) return FDEMRI_ERR_INVALID_ARG;          /* 27-bit row index */
    fdemri_plan_s* p = new (std::nothrow) fdemri_plan_s();
    if (!p) return FDEMRI_ERR_INVALID_ARG;
    p->d.n_modes = n_modes;
    p->d.n_batch = n_batch;
    p->d.n_knots = n_knots;
    p->d.n_seg = n_knots - 1;
    p->d.n_groups = (n_knots - 1 + 31) / 32;
    p->d.ent_max = 3 * 32 * p->d.n_groups;            /* key = vs * ent_max + branch * 32 n_groups + segment */
    p->d.n_freq = n_freq;
    p->d.bin_major = bin_major ? 1 : 0;
    p->d.tile_bins = tile_bins;
    p->d.n_tiles = (int)n_tiles;
    p->d.f0 = f0;
    p->d.df = df;
    p->d.inv_df = (df > 0.0) ? 1.0 / df : 0.0;
    p->d.freq = freq_dev;
    p->d.lut = nullptr;
    /* explicit grids: four buckets per bin (a log-spaced array puts many bins into its lowest buckets), at most 4 M */
    p->d.lut_n = freq_dev ? (int)std::min<int64_t>(4 * n_freq, (int64_t)1 << 22) : 0;
    p->lmn.assign(lmn_host, lmn_host + (size_t)3 * n_modes);
    if (k_host) p->kk.assign(k_host, k_host + n_modes);
    build_weight_table(p);
    p->t_knots_dev = t_knots_dev;
    p->ws = nullptr;
    p->ws_bytes = 0;
    p->built = false;
    p->last_stream = nullptr;
    p->sum_blocks_per_sm = 0;
    p->mode_mask = nullptr;
    p->flags = flags;
    p->ev_valid = false;
    p->ev0 = p->ev1 = nullptr;
    p->side = nullptr;
    p->ev_fork = p->ev_join = nullptr;
    p->lut_built = false;
    p->angle_stage = nullptr;
    p->ev_angles = nullptr;
    p->last_stream_valid = false;
    p->sm_count = prop.multiProcessorCount;
    if (cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_angles, cudaEventDisableTiming) != cudaSuccess ||
        cudaHostAlloc((void**)&p->angle_stage, (size_t)2 * n_batch * sizeof(double), cudaHostAllocDefault) != cudaSuccess) {
        release_plan(p);
        return FDEMRI_ERR_CUDA;
    }
    if (flags & FDEMRI_FLAG_TIMING) {
        if (cudaEventCreate(&p->ev0) != cudaSuccess || cudaEventCreate(&p->ev1) != cudaSuccess) {
            release_plan(p);
            return FDEMRI_ERR_CUDA;
        }
    }
    carve(p, nullptr);
    *out = p;
    return FDEMRI_OK;
}

extern "C" int fdemri_plan(fdemri_plan_t* out, int n_modes, const int32_t* lmn_host, int n_batch, int n_knots,
                           const double* t_knots_dev, int64_t n_freq, const double* freq_dev, double f0, double df,
                           uint32_t flags) {
    return plan_impl(out, n_modes, lmn_host, nullptr, n_batch, n_knots, t_knots_dev, n_freq, freq_dev, f0, df, flags);
}

extern "C" int fdemri_plan_kerr(fdemri_plan_t* out, int n_modes, const int32_t* lmkn_host, int n_batch, int n_knots,
                                const double* t_knots_dev, int64_t n_freq, const double* freq_dev, double f0, double df,
                                uint32_t flags) {
    if (out) *out = nullptr;
    if (!out || !lmkn_host || n_modes < 1 || n_modes > (1 << 20)) return FDEMRI_ERR_INVALID_ARG;
    std::vector<int32_t> lmn((size_t)3 * n_modes), kk(n_modes);
    for (int v = 0; v < n_modes; ++v) {              // (l, m, k, n): the order of Eq. 1's subscript
        lmn[3 * v] = lmkn_host[4 * v];
        lmn[3 * v + 1] = lmkn_host[4 * v + 1];
        kk[v] = lmkn_host[4 * v + 2];
        lmn[3 * v + 2] = lmkn_host[4 * v + 3];
    }
    return plan_impl(out, n_modes, lmn.data(), kk.data(), n_batch, n_knots, t_knots_dev, n_freq, freq_dev, f0, df, flags);
}

extern "C" size_t fdemri_workspace_bytes(fdemri_plan_t p) {
    if (!p) return 0;
    fdemri_plan_s tmp = *p;
    return carve(&tmp, nullptr);
}

extern "C" size_t fdemri_workspace_bytes_min(fdemri_plan_t p) { return fdemri_workspace_bytes(p); }

extern "C" int fdemri_set_workspace(fdemri_plan_t p, void* dev_ptr, size_t bytes) {
    if (!p || !dev_ptr) return FDEMRI_ERR_INVALID_ARG;
    if (((uintptr_t)dev_ptr & 255) != 0) return FDEMRI_ERR_INVALID_ARG;
    fdemri_plan_s tmp = *p;
    const size_t fixed = carve(&tmp, nullptr);
    if (bytes < fixed) return FDEMRI_ERR_WORKSPACE;
    p->ws = dev_ptr;
    p->ws_bytes = bytes;
    carve(p, (char*)dev_ptr);
    p->built = false;
    p->lut_built = false;
    if (cudaMemcpy(p->lmn_dev, p->lmn.data(), p->lmn.size() * sizeof(int32_t), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->lm_index_dev, p->lm_index.data(), p->lm_index.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->wmeta_dev, p->wmeta.data(), p->wmeta.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->wcoef_dev, p->wcoef.data(), p->wcoef.size() * sizeof(double), cudaMemcpyHostToDevice) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    if (p->k_dev && cudaMemcpy(p->k_dev, p->kk.data(), p->kk.size() * sizeof(int32_t), cudaMemcpyHostToDevice) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    if (cudaMemset(p->stats, 0, 16 * sizeof(unsigned long long)) != cudaSuccess) return FDEMRI_ERR_CUDA;
    return FDEMRI_OK;
}

// The dynamic shared memory limit of a kernel is an attribute of the function, per device and process-wide (not per
// plan): set it once per device to what the largest plan (FDEMRI_MAX_KNOTS) can ask for.
static int raise_spline_smem_limits() {
    static bool done[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return FDEMRI_ERR_CUDA;
    if (dev >= 0 && dev < 64 && done[dev]) return FDEMRI_OK;
    const int N = FDEMRI_MAX_KNOTS;
    const size_t sm_sh = (size_t)(2 * N * FDEMRI_SH_ROW + 6 * N) * sizeof(double2);
    const size_t sm_am = ((size_t)2 * N * FDEMRI_AMP_ROW + N + (N & 1)) * sizeof(double) +
                         (size_t)2 * FDEMRI_AMP_VOICES * N * sizeof(double2);
    if (cudaFuncSetAttribute(k_spline_shared<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_sh) != cudaSuccess ||
        cudaFuncSetAttribute(k_spline_shared<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_sh) != cudaSuccess ||
        cudaFuncSetAttribute(k_spline_amp, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_am) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    if (dev >= 0 && dev < 64) done[dev] = true;
    return FDEMRI_OK;
}

static int build_impl(fdemri_plan_t p, const double* f_phi, const double* f_theta, const double* f_r,
                      const double* Phi_phi, const double* Phi_theta, const double* Phi_r, const double* amp,
                      void* cuda_stream) {
    if (!p || !f_phi || !f_r || !Phi_phi || !Phi_r || !amp) return FDEMRI_ERR_INVALID_ARG;
    const bool polar = !p->kk.empty();
    if (polar != (f_theta != nullptr) || polar != (Phi_theta != nullptr)) return FDEMRI_ERR_INVALID_ARG;
    if (!p->ws) return FDEMRI_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const FdemriDims& d = p->d;
    p->last_stream = st;
    if (raise_spline_smem_limits() != FDEMRI_OK) return FDEMRI_ERR_CUDA;
    if (cudaMemsetAsync(p->stats, 0, p->build_clear_bytes, st) != cudaSuccess) return FDEMRI_ERR_CUDA;   /* stats, iband, item_evals */
    if (d.lut && !p->lut_built) {
        // explicit frequency array: its bucket table, once per work space (the lookups check every answer against the
        // array itself, so a table that has gone stale or been overwritten costs time, never a bin)
        k_freq_lut<<<(d.lut_n + 1 + 255) / 256, 256, 0, st>>>(d, const_cast<int*>(d.lut));
        p->lut_built = true;
    }
    // S1: parallel cyclic reduction, one thread per knot.  The amplitude splines (Re/Im A of every voice) are
    // independent of everything S2 needs: they run on the side stream beside the shared splines AND the map, and are
    // joined before the stream goes on (the sum reads them).
    const int N = d.n_knots;
    const int threads = (N + 31) & ~31;
    const size_t sm_sh = (size_t)(2 * N * FDEMRI_SH_ROW + 6 * N) * sizeof(double2);
    const size_t sm_am = ((size_t)2 * N * FDEMRI_AMP_ROW + N + (N & 1)) * sizeof(double) +
                         (size_t)2 * FDEMRI_AMP_VOICES * N * sizeof(double2);
    const int groups = (d.n_modes + FDEMRI_AMP_VOICES - 1) / FDEMRI_AMP_VOICES;
    if (cudaEventRecord(p->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(p->side, p->ev_fork, 0) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    k_spline_amp<<<(unsigned)((size_t)d.n_batch * groups), threads, sm_am, p->side>>>(d.n_modes, N, p->t_knots_dev, amp,
                                                                                   p->rec, p->stats + 5);
    if (cudaEventRecord(p->ev_join, p->side) != cudaSuccess) return FDEMRI_ERR_CUDA;
    // four threads per knot (a component each) up to 256 knots, two above
    if (N <= 256)
        k_spline_shared<4><<<dim3(d.n_batch, polar ? 2 : 1), (4 * N + 31) & ~31, sm_sh, st>>>(
            N, p->t_knots_dev, f_phi, f_r, Phi_phi, Phi_r, p->sh_hi, p->sh_lo, p->stats + 5, f_theta, Phi_theta, p->sh2_hi, p->sh2_lo);
    else
        k_spline_shared<2><<<dim3(d.n_batch, polar ? 2 : 1), (2 * N + 31) & ~31, sm_sh, st>>>(
            N, p->t_knots_dev, f_phi, f_r, Phi_phi, Phi_r, p->sh_hi, p->sh_lo, p->stats + 5, f_theta, Phi_theta, p->sh2_hi, p->sh2_lo);
    // S2: records, entries and their bands: one warp per (batch item, voice)
    const size_t nvoice = (size_t)d.n_batch * d.n_modes;
    auto records = polar ? k_records<true> : k_records<false>;
    records<<<(unsigned)((nvoice + FDEMRI_REC_WARPS - 1) / FDEMRI_REC_WARPS), FDEMRI_REC_WARPS * 32, 0, st>>>(
        d, p->lmn_dev, p->t_knots_dev, p->sh_hi, p->sh_lo, f_phi, f_r, p->rec, p->ent, p->gband, p->vband, p->iband,
        p->mode_mask, p->stats, p->item_evals, p->k_dev, p->sh2_hi, p->sh2_lo, f_theta);
    if (cudaStreamWaitEvent(st, p->ev_join, 0) != cudaSuccess) return FDEMRI_ERR_CUDA;
    if (cudaGetLastError() != cudaSuccess) return FDEMRI_ERR_CUDA;
    p->built = true;
    return FDEMRI_OK;
}

extern "C" int fdemri_build_splines(fdemri_plan_t p, const double* f_phi, const double* f_r, const double* Phi_phi,
                                    const double* Phi_r, const double* amp, void* cuda_stream) {
    return build_impl(p, f_phi, nullptr, f_r, Phi_phi, nullptr, Phi_r, amp, cuda_stream);
}

extern "C" int fdemri_build_splines_kerr(fdemri_plan_t p, const double* f_phi, const double* f_theta, const double* f_r,
                                         const double* Phi_phi, const double* Phi_theta, const double* Phi_r,
                                         const double* amp, void* cuda_stream) {
    if (!f_theta || !Phi_theta) return FDEMRI_ERR_INVALID_ARG;
    return build_impl(p, f_phi, f_theta, f_r, Phi_phi, Phi_theta, Phi_r, amp, cuda_stream);
}

// S0: the viewing angles go through the plan's pinned buffer to the device, then k_weights.  Shared by the sums.
static int stage_weights(fdemri_plan_t p, int n_angles, const double* theta_host, const double* phi_host, cudaStream_t st,
                         bool reset_sum_counters) {
    const FdemriDims& d = p->d;
    for (int i = 0; i < n_angles; ++i)
        if (!std::isfinite(theta_host[i]) || !std::isfinite(phi_host[i])) return FDEMRI_ERR_INVALID_ARG;
    const int nw = n_angles * d.n_modes;
    unsigned long long* counters = reset_sum_counters ? p->stats : nullptr;
    if (n_angles == 1) {
        // one viewing direction for the whole batch: the two angles travel as kernel arguments
        p->last_stream = st;
        k_weights<<<(nw + 127) / 128, 128, 0, st>>>(1, d.n_modes, p->lmn_dev, p->k_dev, p->lm_index_dev, p->wmeta_dev, p->wcoef_dev,
                                                    nullptr, theta_host[0], phi_host[0], p->wts, counters);
        return FDEMRI_OK;
    }
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) return FDEMRI_ERR_CUDA;
    // the pinned staging buffer is read by the asynchronous copy below: wait for the copy of the previous sum
    // (not while a graph is being captured: synchronising is not allowed there)
    if (cap == cudaStreamCaptureStatusNone && p->last_stream_valid && cudaEventSynchronize(p->ev_angles) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    p->last_stream = st;
    for (int i = 0; i < n_angles; ++i) {
        p->angle_stage[2 * i] = theta_host[i];
        p->angle_stage[2 * i + 1] = phi_host[i];
    }
    if (cudaMemcpyAsync(p->angles, p->angle_stage, (size_t)2 * n_angles * sizeof(double), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    // (a stream being captured into a CUDA graph: no event; a replay reads the buffer as the last call left it)
    p->last_stream_valid = cap == cudaStreamCaptureStatusNone && cudaEventRecord(p->ev_angles, st) == cudaSuccess;
    k_weights<<<(nw + 127) / 128, 128, 0, st>>>(n_angles, d.n_modes, p->lmn_dev, p->k_dev, p->lm_index_dev, p->wmeta_dev, p->wcoef_dev,
                                                p->angles, 0.0, 0.0, p->wts, counters);
    return FDEMRI_OK;
}

// S0 + S3 + S4 (+ the fused inner products when inner_out_dev is given)
static int enqueue_sum(fdemri_plan_t p, int n_angles, const double* theta_host, const double* phi_host, double* hplus_dev,
                       double* hcross_dev, const double* weight_dev, const double* dplus_dev, const double* dcross_dev,
                       int hann, double* inner_out_dev, void* cuda_stream) {
    if (!p || !theta_host || !phi_host) return FDEMRI_ERR_INVALID_ARG;
    if ((hplus_dev == nullptr) != (hcross_dev == nullptr)) return FDEMRI_ERR_INVALID_ARG;
    if (!hplus_dev && !inner_out_dev) return FDEMRI_ERR_INVALID_ARG;
    if ((dplus_dev == nullptr) != (dcross_dev == nullptr)) return FDEMRI_ERR_INVALID_ARG;
    if (!p->ws) return FDEMRI_ERR_WORKSPACE;
    if (!p->built) return FDEMRI_ERR_NOT_BUILT;
    const FdemriDims& d = p->d;
    if (n_angles != 1 && n_angles != d.n_batch) return FDEMRI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    {
        // (k_weights also resets the per-sum counters: n_airy, the tile counter, n_slow, n_pairs, the sum's flags)
        const int rc = stage_weights(p, n_angles, theta_host, phi_host, st, true);
        if (rc != FDEMRI_OK) return rc;
    }
    SumArgs a;
    a.d = d;
    a.rec = p->rec;
    a.ent = p->ent;
    a.gband = p->gband;
    a.vband = p->vband;
    a.iband = p->iband;
    a.wts = p->wts;
    a.n_angles = n_angles;
    a.hp = hplus_dev;
    a.hx = hcross_dev;
    a.tile_counter = (unsigned int*)(p->stats + 6);
    a.stats = p->stats;
    a.total_tiles = d.n_tiles * d.n_batch;
    a.weight = weight_dev;
    a.dplus = dplus_dev;
    a.dcross = dcross_dev;
    a.inner_part = inner_out_dev ? p->inner_part : nullptr;
    a.inner_edge = (inner_out_dev && hann) ? p->inner_edge : nullptr;
    const bool bin_major = d.bin_major != 0;
    const size_t smem = bin_major ? sizeof(FdemriBinSmem) : sizeof(FdemriTileSmem);
    const int threads = bin_major ? FDEMRI_BIN_WARPS * 32 : FDEMRI_SUM_THREADS;
    if (p->sum_blocks_per_sm == 0) {
        const void* fn = bin_major ? (const void*)k_bin_sum : (const void*)k_tile_sum;
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return FDEMRI_ERR_CUDA;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, smem) != cudaSuccess || per_sm < 1)
            per_sm = 1;
        p->sum_blocks_per_sm = per_sm;
        if (getenv("FDEMRI_DEBUG"))
            fprintf(stderr, "[fdemri] %s: %d threads, %zu B smem, %d CTAs/SM\n", bin_major ? "k_bin_sum" : "k_tile_sum", threads,
                    smem, per_sm);
    }
    long long grid = (long long)p->sm_count * p->sum_blocks_per_sm;
    if (grid > a.total_tiles) grid = a.total_tiles;
    if (p->ev0) cudaEventRecord(p->ev0, st);
    if (bin_major) k_bin_sum<<<(unsigned)grid, threads, smem, st>>>(a);
    else k_tile_sum<<<(unsigned)grid, threads, smem, st>>>(a);
    if (p->ev1) { cudaEventRecord(p->ev1, st); p->ev_valid = true; }
    {
        const cudaError_t err = cudaGetLastError();
        if (err != cudaSuccess) {
            if (getenv("FDEMRI_DEBUG")) fprintf(stderr, "[fdemri] fdemri_sum: %s\n", cudaGetErrorString(err));
            return FDEMRI_ERR_CUDA;
        }
    }
    if (inner_out_dev) {
        const size_t n_ranges = bin_major ? (size_t)d.n_tiles : (size_t)d.n_tiles * FDEMRI_CWARPS;
        k_inner_reduce<<<d.n_batch, 256, 0, st>>>(n_ranges, bin_major ? d.tile_bins : 32 * FDEMRI_BPL, d.n_freq, p->inner_part,
                                                  a.inner_edge, weight_dev, dplus_dev, dcross_dev, inner_out_dev);
        if (cudaGetLastError() != cudaSuccess) return FDEMRI_ERR_CUDA;
    }
    return FDEMRI_OK;
}

extern "C" int fdemri_td_sum(fdemri_plan_t p, int n_angles, const double* theta_host, const double* phi_host, int64_t n_samples,
                             double t0, double dt, double* hplus_td_dev, double* hcross_td_dev, void* cuda_stream) {
    if (!p || !theta_host || !phi_host || !hplus_td_dev || !hcross_td_dev || n_samples < 1 || !(dt > 0.0) ||
        !std::isfinite(t0) || !std::isfinite(dt))
        return FDEMRI_ERR_INVALID_ARG;
    if (!p->ws) return FDEMRI_ERR_WORKSPACE;
    if (!p->built) return FDEMRI_ERR_NOT_BUILT;
    const FdemriDims& d = p->d;
    if (n_angles != 1 && n_angles != d.n_batch) return FDEMRI_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int rc = stage_weights(p, n_angles, theta_host, phi_host, st, false);
    if (rc != FDEMRI_OK) return rc;
    const dim3 grid((unsigned)((n_samples + 255) / 256), (unsigned)d.n_batch);
    k_td_sum<<<grid, 256, 0, st>>>(d, p->rec, p->t_knots_dev, p->wts, n_angles, p->mode_mask, (long long)n_samples, t0, dt,
                                   hplus_td_dev, hcross_td_dev);
    return cudaGetLastError() == cudaSuccess ? FDEMRI_OK : FDEMRI_ERR_CUDA;
}

extern "C" int fdemri_sum(fdemri_plan_t p, int n_angles, const double* theta_host, const double* phi_host,
                          double* hplus_dev, double* hcross_dev, void* cuda_stream) {
    if (!hplus_dev || !hcross_dev) return FDEMRI_ERR_INVALID_ARG;
    return enqueue_sum(p, n_angles, theta_host, phi_host, hplus_dev, hcross_dev, nullptr, nullptr, nullptr, 0, nullptr, cuda_stream);
}

extern "C" int fdemri_sum_inner(fdemri_plan_t p, int n_angles, const double* theta_host, const double* phi_host,
                                const double* weight_dev, const double* data_plus_dev, const double* data_cross_dev,
                                int hann, double* hplus_dev, double* hcross_dev, double* inner_out_dev, void* cuda_stream) {
    if (!inner_out_dev) return FDEMRI_ERR_INVALID_ARG;
    return enqueue_sum(p, n_angles, theta_host, phi_host, hplus_dev, hcross_dev, weight_dev, data_plus_dev, data_cross_dev,
                       hann, inner_out_dev, cuda_stream);
}


extern "C" int fdemri_select_modes_rule(fdemri_plan_t p, const double* amp_dev, double eps, int rule, unsigned char* keep_dev,
                                        int32_t* n_keep_dev, void* cuda_stream) {
    if (!p || !amp_dev || !keep_dev || !n_keep_dev || !(eps >= 0.0)) return FDEMRI_ERR_INVALID_ARG;
    if (rule != FDEMRI_SELECT_OWN_POWER && rule != FDEMRI_SELECT_CUMULATIVE) return FDEMRI_ERR_INVALID_ARG;
    if (!p->ws) return FDEMRI_ERR_WORKSPACE;
    const FdemriDims& d = p->d;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (rule == FDEMRI_SELECT_OWN_POWER) {
        if (cudaMemsetAsync(n_keep_dev, 0, d.n_batch * sizeof(int32_t), st) != cudaSuccess) return FDEMRI_ERR_CUDA;
        k_select_total<<<d.n_batch * d.n_knots, 256, 0, st>>>(d.n_modes, d.n_knots, amp_dev, p->sel_total);
        const size_t n = (size_t)d.n_batch * d.n_modes;
        k_select_keep<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(d.n_batch, d.n_modes, d.n_knots, amp_dev, p->sel_total, eps,
                                                                   keep_dev, n_keep_dev);
        return cudaGetLastError() == cudaSuccess ? FDEMRI_OK : FDEMRI_ERR_CUDA;
    }
    /* cumulative cut: a sort per (item, time step) in shared memory */
    if (d.n_modes > FDEMRI_SELECT_MAX_MODES) return FDEMRI_ERR_UNSUPPORTED;
    int Vp = 1024;
    while (Vp < d.n_modes) Vp <<= 1;
    const size_t smem = (size_t)Vp * 12 + 1024 * sizeof(double);
    if (cudaFuncSetAttribute(k_select_cumulative, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             FDEMRI_SELECT_MAX_MODES * 12 + 1024 * (int)sizeof(double)) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    if (cudaMemsetAsync(keep_dev, 0, (size_t)d.n_batch * d.n_modes, st) != cudaSuccess) return FDEMRI_ERR_CUDA;
    k_select_cumulative<<<d.n_batch * d.n_knots, 1024, smem, st>>>(d.n_modes, d.n_knots, Vp, amp_dev, eps, keep_dev);
    k_select_count<<<d.n_batch, 256, 0, st>>>(d.n_modes, keep_dev, n_keep_dev);
    return cudaGetLastError() == cudaSuccess ? FDEMRI_OK : FDEMRI_ERR_CUDA;
}

extern "C" int fdemri_select_modes(fdemri_plan_t p, const double* amp_dev, double eps, unsigned char* keep_dev,
                                   int32_t* n_keep_dev, void* cuda_stream) {
    return fdemri_select_modes_rule(p, amp_dev, eps, FDEMRI_SELECT_OWN_POWER, keep_dev, n_keep_dev, cuda_stream);
}

// ---- mode selection for callers that cannot allocate (fdemri.h: fdemri_select_modes_static) ----------------------
// The [n_batch][n_knots] scratch of total powers that fdemri_select_modes keeps in the caller's work space lives here in
// a file-scope device array: every GPU that loads the library holds FDEMRI_STATIC_MAX_TOTALS doubles (256 KB) until the
// process exits.  In host code the array's name is a stand-in of the host side, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) double g_select_total_static[FDEMRI_STATIC_MAX_TOTALS];

static int select_static_scratch(double** out) {
    static std::mutex mu;
    static double* ptr_of_device[FDEMRI_STATIC_MAX_DEVICES] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return FDEMRI_ERR_CUDA;
    if (dev < 0 || dev >= FDEMRI_STATIC_MAX_DEVICES) return FDEMRI_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of_device[dev]) {
        void* q = nullptr;
        if (cudaGetSymbolAddress(&q, g_select_total_static) != cudaSuccess || !q) return FDEMRI_ERR_CUDA;
        ptr_of_device[dev] = static_cast<double*>(q);
    }
    *out = ptr_of_device[dev];
    return FDEMRI_OK;
}

extern "C" int fdemri_select_modes_static(int n_batch, int n_modes, int n_knots, const double* amp_dev, double eps,
                                          unsigned char* keep_dev, int32_t* n_keep_dev, void* cuda_stream) {
    if (n_batch < 1 || n_modes < 1 || n_knots < 1 || !amp_dev || !keep_dev || !n_keep_dev || !(eps >= 0.0))
        return FDEMRI_ERR_INVALID_ARG;
    if ((int64_t)n_batch * n_knots > FDEMRI_STATIC_MAX_TOTALS) return FDEMRI_ERR_STATIC_SCRATCH;
    const size_t n = (size_t)n_batch * n_modes;
    if ((n + 127) / 128 > 0x7fffffffu) return FDEMRI_ERR_INVALID_ARG;
    double* total = nullptr;
    const int rc = select_static_scratch(&total);
    if (rc != FDEMRI_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    /* n_keep is accumulated with atomicAdd and must start at zero; the totals this call reads are all written by
       k_select_total first, so what the last call left in the scratch is never seen */
    if (cudaMemsetAsync(n_keep_dev, 0, (size_t)n_batch * sizeof(int32_t), st) != cudaSuccess) return FDEMRI_ERR_CUDA;
    k_select_total<<<n_batch * n_knots, 256, 0, st>>>(n_modes, n_knots, amp_dev, total);
    k_select_keep<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(n_batch, n_modes, n_knots, amp_dev, total, eps, keep_dev, n_keep_dev);
    return cudaGetLastError() == cudaSuccess ? FDEMRI_OK : FDEMRI_ERR_CUDA;
}

extern "C" int fdemri_set_mode_mask(fdemri_plan_t p, const unsigned char* keep_dev) {
    if (!p) return FDEMRI_ERR_INVALID_ARG;
    p->mode_mask = keep_dev;
    p->built = false;
    return FDEMRI_OK;
}

extern "C" int fdemri_get_stats(fdemri_plan_t p, fdemri_stats* out) {
    if (!p || !out) return FDEMRI_ERR_INVALID_ARG;
    if (!p->ws) return FDEMRI_ERR_WORKSPACE;
    unsigned long long h[16];
    if (cudaStreamSynchronize(p->last_stream) != cudaSuccess) return FDEMRI_ERR_CUDA;
    if (cudaMemcpy(h, p->stats, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) return FDEMRI_ERR_CUDA;
    out->n_items = h[0];
    out->reserved = 0;
    out->n_evals = h[2];
    out->n_turnover = h[3];
    out->n_airy = h[4];
    out->flags = h[5] | h[9];                          /* build flags | flags of the last sum */
    out->n_slow = h[7];
    out->n_pairs = h[8];
    if (out->flags & FDEMRI_BAD_NONFINITE) return FDEMRI_ERR_INVALID_ARG;
    return FDEMRI_OK;
}

extern "C" int fdemri_get_item_evals(fdemri_plan_t p, uint64_t* out_host) {
    if (!p || !out_host) return FDEMRI_ERR_INVALID_ARG;
    if (!p->ws) return FDEMRI_ERR_WORKSPACE;
    if (!p->built) return FDEMRI_ERR_NOT_BUILT;
    if (cudaStreamSynchronize(p->last_stream) != cudaSuccess) return FDEMRI_ERR_CUDA;
    if (cudaMemcpy(out_host, p->item_evals, (size_t)p->d.n_batch * sizeof(uint64_t), cudaMemcpyDeviceToHost) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    return FDEMRI_OK;
}

// amp_coef[b][v][c][k][j] <- rec[b][v][k][R_AR + 4c + j]
__global__ void k_gather_amp(size_t total, int S, const double* __restrict__ rec, double* __restrict__ out) {
    size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= total) return;
    int j = (int)(id & 3);
    size_t r = id >> 2;
    int k = (int)(r % S);
    r /= S;
    int c = (int)(r & 1);
    size_t bv = r >> 1;
    out[id] = rec[(bv * S + k) * R_DOUBLES + (c ? R_AI : R_AR) + j];
}

extern "C" int fdemri_get_coeffs(fdemri_plan_t p, double* shared_hi_dev, double* shared_lo_dev, double* amp_coef_dev) {
    if (!p) return FDEMRI_ERR_INVALID_ARG;
    if (!p->ws) return FDEMRI_ERR_WORKSPACE;
    if (!p->built) return FDEMRI_ERR_NOT_BUILT;
    const FdemriDims& d = p->d;
    cudaStream_t st = p->last_stream;
    size_t nsh = (size_t)d.n_batch * 4 * d.n_seg * 4 * sizeof(double);
    if (shared_hi_dev && cudaMemcpyAsync(shared_hi_dev, p->sh_hi, nsh, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    if (shared_lo_dev && cudaMemcpyAsync(shared_lo_dev, p->sh_lo, nsh, cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        return FDEMRI_ERR_CUDA;
    if (amp_coef_dev) {
        size_t total = (size_t)d.n_batch * d.n_modes * 2 * d.n_seg * 4;
        k_gather_amp<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(total, d.n_seg, p->rec, amp_coef_dev);
        if (cudaGetLastError() != cudaSuccess) return FDEMRI_ERR_CUDA;
    }
    return FDEMRI_OK;
}

extern "C" int fdemri_get_kernel_ms(fdemri_plan_t p, float* ms_out) {
    if (!p || !ms_out) return FDEMRI_ERR_INVALID_ARG;
    if (!p->ev0 || !p->ev_valid) return FDEMRI_ERR_NOT_BUILT;
    if (cudaEventSynchronize(p->ev1) != cudaSuccess) return FDEMRI_ERR_CUDA;
    if (cudaEventElapsedTime(ms_out, p->ev0, p->ev1) != cudaSuccess) return FDEMRI_ERR_CUDA;
    return FDEMRI_OK;
}

// 8 independent DFMA chains per thread, all in registers.  REG3 = false: a <- a*m + c with loop-invariant m, c (one
// fresh register operand per instruction: the classic peak loop).  REG3 = true: a_i <- a_i*b_i + b_j with three
// distinct, changing register operands -- the form of most DFMAs of a real kernel; on B200 this issues every
// three cycles per SM sub-partition instead of every two (register-file read bandwidth).
template <bool REG3>
__global__ void __launch_bounds__(512) k_dfma_peak(int n_iters, double seed, double* sink) {
    double a[8], b[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = seed + threadIdx.x + i; b[i] = 0.999999 + 1e-9 * (threadIdx.x + i); }
    const double m = 0.999999, c = 1e-9;
    for (int it = 0; it < n_iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = REG3 ? fma(a[i], b[i], b[(i + 3) & 7]) : fma(a[i], m, c);
    }
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) r += a[i];
    if (r == 12345.678) sink[0] = r;     // never true; keeps the chains alive
}

template <bool REG3>
static int measure_peak(int n_iters, double* tflops_out) {
    if (!tflops_out || n_iters < 1) return FDEMRI_ERR_INVALID_ARG;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return FDEMRI_ERR_CUDA;
    double* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return FDEMRI_ERR_CUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int threads = 512, blocks = prop.multiProcessorCount * 4;
    k_dfma_peak<REG3><<<blocks, threads>>>(n_iters / 8 + 1, 1.0, sink);    // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        k_dfma_peak<REG3><<<blocks, threads>>>(n_iters, 1.0, sink);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess) return FDEMRI_ERR_CUDA;
    double flops = 2.0 * 8.0 * (double)n_iters * threads * (double)blocks;
    *tflops_out = flops / (best * 1e-3) * 1e-12;
    return FDEMRI_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Issue-cost microbenchmarks (profiles/r2_dispatch_model.md): 8 independent chains per thread, 16 warps per SM
// sub-partition; the measured quantity is the time per group of instructions per warp and sub-partition, in ns.
//   0  DFMA a_i <- a_i * m + c            one distinct register operand, two shared ones (.reuse)
//   1  DFMA a_i <- a_i * b_i + c          two distinct register operands, one shared
//   2  DFMA a_i <- a_i * b_i + const-bank two distinct register operands and a constant-bank operand
//   3  DFMA a_i <- a_i * b_i + b_j        three distinct register operands
//   4  DMUL a_i <- a_i * b_i              5  DADD a_i <- a_i + b_i
//   6  variant 1 + two integer instructions (xor, add) per DFMA
//   7  variant 1 + four integer instructions per DFMA
//   8  variant 0 + one FFMA (one distinct register operand) per DFMA
//   9  variant 3 + one FFMA (one distinct register operand) per DFMA
// ---------------------------------------------------------------------------------------------------------
__constant__ double c_issue_k[2] = {0.999999, 1e-9};

template <int V>
__global__ void __launch_bounds__(512) k_issue(int n_iters, double seed, double* sink) {
    double a[8], b[8];
    float fa[8];
    int ia[8], ib[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i] = seed + threadIdx.x + i; b[i] = 0.999999 + 1e-9 * (threadIdx.x + i); fa[i] = (float)a[i];
        ia[i] = threadIdx.x * (i + 3); ib[i] = threadIdx.x + i * 7;
    }
    const double m = 0.999999 + seed * 1e-12, c = 1e-9 + seed * 1e-13;
    const float fm = (float)m, fc = (float)c;
    for (int it = 0; it < n_iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (V == 0 || V == 8) a[i] = fma(a[i], m, c);
            if (V == 1 || V == 6 || V == 7) a[i] = fma(a[i], b[i], c);
            if (V == 2) a[i] = fma(a[i], b[i], c_issue_k[1]);
            if (V == 3 || V == 9) a[i] = fma(a[i], b[i], b[(i + 3) & 7]);
            if (V == 4) a[i] = a[i] * b[i];
            if (V == 5) a[i] = a[i] + b[i];
            if (V == 6 || V == 7) ia[i] = (ia[i] ^ ib[i]) + 1;
            if (V == 7) ib[i] = (ib[i] & ia[i]) | 5;
            if (V == 8 || V == 9) fa[i] = fmaf(fa[i], fm, fc);
        }
    }
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) r += a[i] + b[i] + (double)fa[i] + (double)(ia[i] + ib[i]);
    if (r == 12345.678) sink[0] = r;     // never true; keeps the chains alive
}

template <int V>
static int run_issue(int n_iters, double* ns_out) {
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return FDEMRI_ERR_CUDA;
    double* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return FDEMRI_ERR_CUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int threads = 512, per_sm = 4, blocks = prop.multiProcessorCount * per_sm;
    k_issue<V><<<blocks, threads>>>(n_iters / 8 + 1, 1.0, sink);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        k_issue<V><<<blocks, threads>>>(n_iters, 1.0, sink);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess) return FDEMRI_ERR_CUDA;
    // groups issued per sub-partition: 8 per iteration and warp, threads / 32 * per_sm / 4 warps per sub-partition
    const double groups = 8.0 * (double)n_iters * (threads / 32) * per_sm / 4.0;
    *ns_out = (double)best * 1e6 / groups;
    return FDEMRI_OK;
}

extern "C" int fdemri_measure_issue_ns(int variant, int n_iters, double* ns_out) {
    if (!ns_out || n_iters < 1) return FDEMRI_ERR_INVALID_ARG;
    switch (variant) {
        case 0: return run_issue<0>(n_iters, ns_out);
        case 1: return run_issue<1>(n_iters, ns_out);
        case 2: return run_issue<2>(n_iters, ns_out);
        case 3: return run_issue<3>(n_iters, ns_out);
        case 4: return run_issue<4>(n_iters, ns_out);
        case 5: return run_issue<5>(n_iters, ns_out);
        case 6: return run_issue<6>(n_iters, ns_out);
        case 7: return run_issue<7>(n_iters, ns_out);
        case 8: return run_issue<8>(n_iters, ns_out);
        case 9: return run_issue<9>(n_iters, ns_out);
        default: return FDEMRI_ERR_INVALID_ARG;
    }
}

extern "C" int fdemri_measure_fp64_peak(int n_iters, double* tflops_out) { return measure_peak<false>(n_iters, tflops_out); }
extern "C" int fdemri_measure_fp64_peak_3reg(int n_iters, double* tflops_out) { return measure_peak<true>(n_iters, tflops_out); }

extern "C" int fdemri_destroy(fdemri_plan_t p) {
    if (!p) return FDEMRI_ERR_INVALID_ARG;
    release_plan(p);
    return FDEMRI_OK;
}

extern "C" const char* fdemri_strerror(int status) {
    switch (status) {
        case FDEMRI_OK: return "ok";
        case FDEMRI_ERR_INVALID_ARG: return "invalid argument";
        case FDEMRI_ERR_WORKSPACE: return "work space missing or too small";
        case FDEMRI_ERR_CUDA: return "CUDA error";
        case FDEMRI_ERR_NOT_BUILT: return "splines not built";
        case FDEMRI_ERR_UNSUPPORTED: return "call not available in this configuration";
        case FDEMRI_ERR_STATIC_SCRATCH: return "size beyond the library's static scratch (n_batch * n_knots > FDEMRI_STATIC_MAX_TOTALS)";
        default: return "unknown status";
    }
}

extern "C" const char* fdemri_version(void) { return "fdemri 0.1 sm_100a"; }
