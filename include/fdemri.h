/* fdemri.h -- C ABI of libfdemri: the frequency-domain EMRI harmonic sum of arXiv:2307.12585 on one
 * NVIDIA B200 (sm_100a), FP64.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md of the build; see DESIGN.md for the readings):
 *   S1  not-a-knot cubic splines of f_phi, f_r, Phi_phi, Phi_r and of Re/Im A_lmn over the sparse
 *       trajectory;
 *   S2  per voice (l,m,n) and segment, the cubic  f = A + B tau + C tau^2 + D tau^3  (Eq. 6) and
 *       the contiguous range of frequency bins it covers, "predetermined before the summation" (L105), with two
 *       levels of bands over those ranges from which the sum kernels find the entries that meet a tile of bins;
 *   S3  per bin and root t_j(f) the term of Eq. 9 (L107-119):
 *         A(t) g(X)/sqrt|Fdot| exp{i[2 pi f t - Phi(t)]},  X = 2 pi Fdot^3 / (3 Fddot^2),
 *       summed over voices with the spin-weighted harmonics (Eq. 1) into h~+(f), h~x(f), the
 *       (l,-m,-n) partner of every m>0 voice taken from the symmetry A -> (-1)^l conj A;
 *   S4  one coalesced store per bin (no atomics; the paper's kernel adds atomically, L121).
 *
 * Conventions
 *   - "dev" pointers are CUDA device pointers, "host" pointers are host pointers.  The caller owns every
 *     buffer, including the work space; the plan owns only small host metadata.
 *   - No call allocates device memory except the fdemri_measure_* microbenchmarks (8 bytes, freed before they
 *     return); a plan owns a small pinned host buffer (fdemri_select_modes_static needs neither plan nor work space).  build_splines / sum do not synchronise: they enqueue
 *     kernels on `cuda_stream` (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *     build_splines runs one of its kernels on a stream of the plan, forked from and joined back into
 *     `cuda_stream` with events, so ordering on `cuda_stream` is all a caller needs.
 *   - Every function returns a status: 0 = FDEMRI_OK, >0 = error.  No exceptions, no printing (with the
 *     environment variable FDEMRI_DEBUG set, fdemri_sum reports its launch shape and CUDA error strings on stderr).
 *   - Asynchronous CUDA errors surface in the next call or in fdemri_get_stats (which synchronises).
 */
#ifndef FDEMRI_H
#define FDEMRI_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
    FDEMRI_OK = 0,
    FDEMRI_ERR_INVALID_ARG = 1, /* bad size, NULL pointer, l<2, m<0, m>l, unsorted knots ...            */
    FDEMRI_ERR_WORKSPACE = 2,   /* work space missing or smaller than fdemri_workspace_bytes                        */
    FDEMRI_ERR_CUDA = 3,        /* a CUDA runtime call or kernel failed                                   */
    FDEMRI_ERR_NOT_BUILT = 4,   /* fdemri_sum / get_coeffs before fdemri_build_splines                    */
    FDEMRI_ERR_UNSUPPORTED = 5, /* the call is not available in this configuration                                 */
    FDEMRI_ERR_STATIC_SCRATCH = 6 /* fdemri_select_modes_static: n_batch * n_knots > FDEMRI_STATIC_MAX_TOTALS         */
};

/* plan flags */
enum {
    FDEMRI_FLAG_NONE = 0,
    FDEMRI_FLAG_TIMING = 1,    /* record CUDA events around the S3 sum kernel of every fdemri_sum (see
                                  fdemri_get_kernel_ms); costs two event records per call                  */
    FDEMRI_FLAG_BIN_MAJOR = 2, /* force the bin-major sum kernel (a CTA owns 8, 16 or 32 consecutive bins, one warp per bin at a
                                  time, lanes over the entries that cover it): the right shape when a (voice, segment)
                                  covers only a few bins -- sparse or down-sampled frequency arrays (PAPER.md 3.3)   */
    FDEMRI_FLAG_TILE_MAJOR = 4 /* force the tile-major sum kernel (a CTA owns 960 consecutive bins): dense grids.
                                  Default: bin-major iff n_freq < 256 (n_knots - 1)                         */
};

/* bits of fdemri_stats.flags (device-side validation, read back by fdemri_get_stats) */
enum {
    FDEMRI_BAD_TWO_EXTREMA = 1,   /* (kept for ABI stability, never raised: a segment cubic with two interior extrema --
                                     the paper assumes at most one, L105 -- is split into its three monotone branches) */
    FDEMRI_BAD_NONFINITE = 4,     /* NaN/Inf met in the inputs or spline coefficients                      */
    FDEMRI_BAD_NEWTON = 8,        /* a root iteration of the last fdemri_sum hit its iteration cap          */
    FDEMRI_BAD_LIST_OVERFLOW = 16 /* (kept for ABI stability, never raised: there is no work list any more)  */
};

typedef struct fdemri_plan_s* fdemri_plan_t;

typedef struct {
    uint64_t n_items;        /* non-empty (voice, sign, segment-branch) entries of the last build (S2)        */
    uint64_t reserved;
    uint64_t n_evals;        /* "mode-bin evaluations": (voice, sign, root, bin) terms the MAP of the last build assigns,
                                i.e. the sum of the widths of the entries' bin intervals (P9).  Counted in S2, not by
                                the sum kernel: per-bin parity is what shows that every one of them was accumulated
                                (bin-major plans also count the accumulated terms themselves, see n_pairs)           */
    uint64_t n_turnover;     /* segments with an interior extremum of F (Fdot = 0, L92, L105)                 */
    uint64_t n_airy;         /* evaluations that took the small-|X| (Airy) path                              */
    uint64_t flags;          /* OR of FDEMRI_BAD_*                                                            */
    uint64_t n_slow;         /* evaluations of monotone segments that left the fast path (small |X| or a
                                rejected iteration) and took the safeguarded Newton with a division           */
    uint64_t n_pairs;        /* last fdemri_sum: tile-major plans: (entry, tile) pairs the producer warps staged;
                                bin-major plans: terms accumulated (= n_evals)                                   */
} fdemri_stats;

/* Create a plan.
 *  lmn_host    [n_modes][3] int32 (l, m, n) with l >= 2, 0 <= m <= l; copied.  The partner (l,-m,-n) of every
 *              m > 0 voice is implied (L64-66 + symmetry); m = 0 voices stand for themselves.
 *  n_batch     number of independent parameter sets evaluated per call (>= 1)
 *  n_knots     points of the sparse trajectory (4..512), the same for every batch item (L58: ~100)
 *  t_knots_dev [n_batch][n_knots] seconds, strictly increasing; borrowed for the plan's life (every
 *              fdemri_build_splines reads it again, from kernels that run after the call has returned)
 *  n_freq      number of frequency bins
 *  freq_dev    [n_freq] Hz, sorted ascending, >= 0, shared by the batch; borrowed for the plan's life.
 *              NULL selects the uniform grid  f_i = f0 + (double)i*df  (product rounded, then sum rounded) --
 *              with f0 = 0, df = 1/T the DFT grid of L141.
 */
int fdemri_plan(fdemri_plan_t* out, int n_modes, const int32_t* lmn_host, int n_batch, int n_knots,
                const double* t_knots_dev, int64_t n_freq, const double* freq_dev, double f0, double df,
                uint32_t flags);

/* Device work space the plan needs (bytes); the caller allocates it (256-byte aligned) and hands it over.
 * The work space holds the plan's tables (written by fdemri_set_workspace), the spline records, the segment->bin map
 * and its bands; it must stay valid and untouched from fdemri_set_workspace to the last sum.  A plan with an explicit
 * frequency array also keeps a bucket table of that array there, written by the first fdemri_build_splines after
 * fdemri_set_workspace: every lookup through it is checked against the array itself, so changing the array later
 * costs time, never a bin.  fdemri_set_workspace returns FDEMRI_ERR_WORKSPACE for a smaller buffer;
 * it may be called again with another buffer, fdemri_build_splines must then be repeated.
 * One stream at a time: the per-call scratch (angles, weights, counters, partial inner products) lives in the work
 * space, so two fdemri_sum calls on one plan must not run concurrently on different streams. */
size_t fdemri_workspace_bytes(fdemri_plan_t plan);
/* The same number (kept for ABI stability: there is no optional part any more). */
size_t fdemri_workspace_bytes_min(fdemri_plan_t plan);
int fdemri_set_workspace(fdemri_plan_t plan, void* dev_ptr, size_t bytes);

/* S1 + S2 (splines, then the records and the segment->bin map).  All inputs are device pointers, borrowed until the
 * enqueued kernels have run.
 *  f_phi, f_r      [n_batch][n_knots] Hz      fundamental frequencies Omega/(2 pi M) at the knots (L94)
 *  Phi_phi, Phi_r  [n_batch][n_knots] rad     fundamental phases at the knots (L56)
 *  amp             [n_batch][n_modes][n_knots][2] (re, im) mode amplitudes at the knots (L60), with mu/d_L of
 *                  Eq. 1 folded in by the caller */
int fdemri_build_splines(fdemri_plan_t plan, const double* f_phi, const double* f_r, const double* Phi_phi,
                         const double* Phi_r, const double* amp, void* cuda_stream);

/* General voices (l, m, k, n) of Eq. 1 (phase m Phi_phi + k Phi_theta + n Phi_r; L60 "m, k, and n label
 * the azimuthal, polar, and radial modes"; L252: the extension to Kerr the paper announces, "where the number of modes
 * is expected to increase by an order of magnitude").  Same path with a third fundamental frequency:
 *   F_v = m f_phi + k f_theta + n f_r  (knot values rounded in that order),  Phi_v likewise;
 *   the partner (l,-m,-k,-n) of an m > 0 voice is implied with amplitude (-1)^(l+k) conj A  (R16);
 *   the harmonics stay the spin-weighted SPHERICAL ones -- the time-dependent spheroidal harmonics of Kerr are what
 *   the paper leaves to "future work" (L66) and are not part of this library.
 *  lmkn_host   [n_modes][4] int32 (l, m, k, n), l >= 2, 0 <= m <= l; everything else as fdemri_plan.
 * A plan made here is built with fdemri_build_splines_kerr (fdemri_build_splines returns FDEMRI_ERR_INVALID_ARG, and
 * vice versa); every other call is shared.  With k = 0 on every voice the results equal fdemri_plan's bit for bit. */
int fdemri_plan_kerr(fdemri_plan_t* out, int n_modes, const int32_t* lmkn_host, int n_batch, int n_knots,
                     const double* t_knots_dev, int64_t n_freq, const double* freq_dev, double f0, double df,
                     uint32_t flags);
/*  f_theta, Phi_theta  [n_batch][n_knots]  polar fundamental frequency (Hz) and phase (rad) at the knots (L48, L56) */
int fdemri_build_splines_kerr(fdemri_plan_t plan, const double* f_phi, const double* f_theta, const double* f_r,
                              const double* Phi_phi, const double* Phi_theta, const double* Phi_r, const double* amp,
                              void* cuda_stream);

/* S0 + S3 + S4 (S2 is part of fdemri_build_splines).
 *  theta_host, phi_host  source-frame viewing angles (L66), [n_angles] on the host, n_angles = 1 or n_batch; read
 *                        before the call returns.  n_angles = 1: the pair travels as kernel arguments (a call captured
 *                        into a CUDA graph replays the angles of the capture).  n_angles = n_batch: copied through a
 *                        pinned buffer of the plan (a replay uses the angles of the most recent such call on the plan).
 *  hplus_dev, hcross_dev [n_batch][n_freq][2] (re, im) FP64, fully overwritten (zeros where no voice has
 *                        support, L147; the bin f = 0 is always zero) */
int fdemri_sum(fdemri_plan_t plan, int n_angles, const double* theta_host, const double* phi_host,
               double* hplus_dev, double* hcross_dev, void* cuda_stream);

/* S0 + S3 + S4 with the noise-weighted inner products of Eq. 12 (the likelihood of Eq. 13,
 * L151-153) accumulated on the fly, so that the waveform need not be written to memory:
 *     <a|b> = sum_k w_k [ a+(f_k) conj b+(f_k) + ax(f_k) conj bx(f_k) ]
 * (the paper's inner product is the real part with w_k = 4 df / S_n(f_k); ln L = -(<d|d> - 2 Re<d|h> + <h|h>)/2).
 *  weight_dev     [n_freq] w_k >= 0, shared by the batch; NULL: w = 1
 *  data_plus_dev, data_cross_dev  [n_freq][2] (re, im) data of the two polarisations, shared by the batch; both
 *                 NULL: only <h|h> is formed
 *  hann           != 0: the waveform entering the inner products is first convolved with the DFT of the Hann
 *                 window, h_k/2 - h_{k-1}/4 - h_{k+1}/4 with bins outside the grid counting as zero (L145: the
 *                 window the paper applies to the time series); the waveform written to hplus/hcross is not filtered
 *  hplus_dev, hcross_dev  as in fdemri_sum, or both NULL: nothing but the inner products leaves the kernel
 *                 (either sum kernel)
 *  inner_out_dev  [n_batch][4] = {<h|h>, Re<d|h>, Im<d|h>, 0}, device memory; sums are formed in a fixed order
 *                 (bitwise reproducible) */
int fdemri_sum_inner(fdemri_plan_t plan, int n_angles, const double* theta_host, const double* phi_host,
                     const double* weight_dev, const double* data_plus_dev, const double* data_cross_dev, int hann,
                     double* hplus_dev, double* hcross_dev, double* inner_out_dev, void* cuda_stream);

/* The time-domain voice sum of Eq. 1 / Eq. 2 from the splines of the last
 * fdemri_build_splines: the signal whose Fourier transform (Eq. 3) the stationary-phase sum of fdemri_sum
 * approximates, on the uniform time grid t_j = t0 + (double)j * dt, j = 0 .. n_samples - 1:
 *     h(t) = h+ - i hx = sum_v A_v(t) Y_lm e^{-i Phi_v(t)}  +  [m > 0]  (-1)^(l+k) conj(A_v(t)) Y_l,-m e^{+i Phi_v(t)}.
 * Samples outside [t_0, t_{N-1}) of the batch item's trajectory are 0.  Modes dropped by fdemri_set_mode_mask are
 * left out.  (With N_s samples and Delta t = dt:  h~+(f_i) ~ N_s dt ifft(h+)_i  for f_i = i / (N_s dt): the sign
 * convention of Eq. 3.)
 *  theta_host, phi_host      as in fdemri_sum
 *  hplus_td_dev, hcross_td_dev  [n_batch][n_samples] real FP64, fully overwritten
 * One thread per sample, all voices in list order: the work is n_samples x n_modes (the paper's time-domain cost, L210). */
int fdemri_td_sum(fdemri_plan_t plan, int n_angles, const double* theta_host, const double* phi_host, int64_t n_samples,
                  double t0, double dt, double* hplus_td_dev, double* hcross_td_dev, void* cuda_stream);

/* Mode selection by power threshold: per time step of the sparse trajectory the
 * modes are sorted by |A_lmkn(t)|^2 in descending order, a cumulative sum is formed, and the modes whose "additional
 * power" stays above "the threshold eps related to the total power emitted" contribute; "the selected modes are given
 * by the union of all contributing modes across all time steps".  The rule itself is not printed (the paper defers to
 * Katz et al. 2021): both readings of DESIGN.md R15 are available.
 *   FDEMRI_SELECT_OWN_POWER   a mode contributes at a time step iff |A|^2 >= eps * (sum over all modes of |A|^2 there);
 *   FDEMRI_SELECT_CUMULATIVE  the contributing modes are the shortest prefix of the sorted array whose cumulative sum
 *                             reaches (1 - eps) * total: the discarded power is at most eps * total per time step
 *                             (a sort per (item, time step) in shared memory: n_modes <= 16384, else
 *                             FDEMRI_ERR_UNSUPPORTED).
 *  amp_dev     [n_batch][n_modes][n_knots][2], as in fdemri_build_splines
 *  eps         >= 0
 *  keep_dev    [n_batch][n_modes] bytes, out: 1 = selected
 *  n_keep_dev  [n_batch] int32, out: number of selected modes
 * Needs the work space (a [n_batch][n_knots] scratch of total powers).  Enqueued on cuda_stream.
 * fdemri_select_modes is fdemri_select_modes_rule with FDEMRI_SELECT_OWN_POWER. */
enum { FDEMRI_SELECT_OWN_POWER = 0, FDEMRI_SELECT_CUMULATIVE = 1 };
int fdemri_select_modes_rule(fdemri_plan_t plan, const double* amp_dev, double eps, int rule, unsigned char* keep_dev,
                             int32_t* n_keep_dev, void* cuda_stream);
int fdemri_select_modes(fdemri_plan_t plan, const double* amp_dev, double eps, unsigned char* keep_dev,
                        int32_t* n_keep_dev, void* cuda_stream);
/* fdemri_select_modes (FDEMRI_SELECT_OWN_POWER) for callers that cannot allocate device memory or hold a plan: code
 * between other work under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No plan, no work
 * space: the [n_batch][n_knots] scratch of total powers is a static device array inside the library
 * (FDEMRI_STATIC_MAX_TOTALS doubles = 256 KB, held by every GPU that loads the library until the process exits).  The
 * call allocates nothing on the device or the host (no cudaMalloc / cudaFree / cudaHostAlloc, no plan): its first use
 * on a device asks the runtime for the array's address, later calls only enqueue one memset of n_keep_dev and two
 * kernels on cuda_stream.
 *  n_batch, n_modes, n_knots  >= 1;  n_batch * n_knots <= FDEMRI_STATIC_MAX_TOTALS, else FDEMRI_ERR_STATIC_SCRATCH
 *                             (nothing is enqueued); devices with ordinal >= FDEMRI_STATIC_MAX_DEVICES:
 *                             FDEMRI_ERR_UNSUPPORTED
 *  amp_dev, eps, keep_dev, n_keep_dev, cuda_stream   as in fdemri_select_modes; results are bit-identical to it.
 * Every call on a device shares the one array, which keeps the last call's totals (a call overwrites all it reads, so
 * nothing has to be cleared but n_keep_dev, which the call clears): two calls that overlap on the GPU -- different
 * streams, or the same graph launched twice concurrently -- race.  Serialise them (one stream, or events). */
enum { FDEMRI_STATIC_MAX_TOTALS = 32768, FDEMRI_STATIC_MAX_DEVICES = 64 };
int fdemri_select_modes_static(int n_batch, int n_modes, int n_knots, const double* amp_dev, double eps,
                               unsigned char* keep_dev, int32_t* n_keep_dev, void* cuda_stream);
/* Modes with keep_dev[b][v] == 0 get no entries in the next fdemri_build_splines and so never reach the sum.
 * keep_dev is borrowed until it is replaced or the plan is destroyed (every later build reads it, from a kernel that
 * runs after the call has returned); NULL: every mode of the list is summed.  The mode list of the plan is unchanged. */
int fdemri_set_mode_mask(fdemri_plan_t plan, const unsigned char* keep_dev);

/* Counters of the last fdemri_build_splines / fdemri_sum (synchronises the stream used by the last call). */
int fdemri_get_stats(fdemri_plan_t plan, fdemri_stats* out);
/* fdemri_stats.n_evals per batch item: out_host [n_batch] on the host.  Synchronises like fdemri_get_stats. */
int fdemri_get_item_evals(fdemri_plan_t plan, uint64_t* out_host);

/* Spline coefficients as built on the device, for parity level A (oracle fed the GPU's coefficients).
 *  shared_hi, shared_lo [n_batch][4][n_knots-1][4]  (a,b,c,d) of f_phi, f_r, Phi_phi, Phi_r as hi + lo doubles
 *  amp_coef             [n_batch][n_modes][2][n_knots-1][4]  (a,b,c,d) of Re A, Im A
 * Device pointers; any may be NULL.  Enqueued on the stream of the last build_splines.  (A plan of general voices
 * returns the same four shared components; the splines of f_theta, Phi_theta stay in the work space.) */
int fdemri_get_coeffs(fdemri_plan_t plan, double* shared_hi_dev, double* shared_lo_dev, double* amp_coef_dev);

/* Device time in ms of the S3/S4 tile kernel of the last fdemri_sum, from CUDA events recorded on that call's
 * stream (plan created with FDEMRI_FLAG_TIMING).  Synchronises on the stop event. */
int fdemri_get_kernel_ms(fdemri_plan_t plan, float* ms_out);

/* FP64 FMA peak of the current device measured with a register-resident DFMA loop (the roofline denominator
 * of the ALU-bound tile kernel): writes TFLOP/s (2 flop per DFMA).  Synchronous; n_iters ~ 1<<16. */
int fdemri_measure_fp64_peak(int n_iters, double* tflops_out);
/* The same loop with three distinct, changing register operands per DFMA (a_i <- a_i*b_i + b_j): the rate a
 * general FP64 kernel can reach; on B200 about 2/3 of the figure above (register-file read bandwidth). */
int fdemri_measure_fp64_peak_3reg(int n_iters, double* tflops_out);

/* Issue-cost microbenchmarks behind the roofline discussion of DESIGN.md (what an FP64 instruction costs on a B200
 * sub-partition as a function of its distinct register operands, and whether integer / FP32 instructions issue in its
 * shadow).  variant 0..9: see csrc/fdemri.cu; ns_out = time per group of instructions per warp and sub-partition.
 * Synchronous; n_iters ~ 1 << 15. */
int fdemri_measure_issue_ns(int variant, int n_iters, double* ns_out);

int fdemri_destroy(fdemri_plan_t plan);
const char* fdemri_strerror(int status);
/* Library version string, e.g. "fdemri 0.1 sm_100a". */
const char* fdemri_version(void);

#ifdef __cplusplus
}
#endif
#endif
