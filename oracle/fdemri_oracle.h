/* fdemri_oracle.h -- CPU oracle for the frequency-domain EMRI harmonic sum of arXiv:2307.12585.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2307_12585_b200/) may include, link
 * or call this.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs use it.  It shares no code with the CUDA library.
 *
 * Plain, slow, step-by-step: long double arithmetic on the given double inputs, in the paper's order
 *   splines  ->  per voice/segment cubic f = A+B tau+C tau^2+D tau^3 (Eq. 6)
 *   ->  real roots inside the segment (L105)  ->  Eq. 9 term per root (L107-119, read as DESIGN.md R3/R4)
 *   ->  sum over voices into h+ and hx (Eq. 1-3; L66 for the polarisations).
 * All pointers are HOST pointers.  All functions return 0 on success, >0 on invalid arguments.
 *
 * Pins (tests/test_oracle_*.py): P1 spline vs cubic reproduction and scipy not-a-knot; P2 -2Y_lm closed
 * forms / orthonormality; P3 linear-chirp closed-form SPA; P4 quadratic chirp = Airy closed form; P5 g(X) vs
 * mpmath Hankel + Eq. 8 quadrature; P6 brute-force FFT of the time-domain sum; P7 (l,-m,-n) symmetry;
 * P8 zero outside support and root counts.  Unpinned: the paper's own K_{1/3} polynomial coefficients and
 * FEW's actual output values (not printed in the paper; no code) -- "parity unpinned" for those only.
 */
#ifndef FDEMRI_ORACLE_H
#define FDEMRI_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* O1 (L60): not-a-knot cubic spline coefficients of n_comp components on shared knots t[n_knots].
 * y: [n_comp][n_knots].  Output coefficient (a,b,c,d) of segment k, tau = t - t_k, as hi + lo doubles
 * (hi = (double)x, lo = (double)(x - hi); together they hold the long double exactly):
 * coef_hi, coef_lo: [n_comp][n_knots-1][4].  coef_lo may be NULL. */
int fdemri_oracle_build_splines(int n_knots, const double* t, int n_comp, const double* y,
                                double* coef_hi, double* coef_lo);

/* Spin-weight -2 spherical harmonic -2Y_lm(theta, phi) (L66; Goldberg et al. sum). */
int fdemri_oracle_ylm(int l, int m, double theta, double phi, double* re, double* im);

/* g(X) of DESIGN.md R3/R4: sqrt(pi|X|/2) e^{i pi/6} e^{-i|X|} H^(1)_{1/3}(|X|) for X>0, conjugate for X<0. */
int fdemri_oracle_g(double X, double* re, double* im);
/* g(X)/sqrt|Fdot| with X = 2 pi Fdot^3/(3 Fddot^2), regular at Fdot -> 0 (Airy form).  Returns 1 if
 * Fdot = Fddot = 0 (no term, R10). */
int fdemri_oracle_g_over_sqrt(double Fdot, double Fddot, double* re, double* im);

/* The harmonic sum (O2, O3) from given spline coefficients.
 *  lmn          [n_modes][3] (l,m,n), m >= 0 (partner (l,-m,-n) implied for m>0, R1)
 *  t            [n_knots] knot times, strictly increasing
 *  fphi_k, fr_k [n_knots] knot values of f_phi, f_r in Hz (decide membership, R6)
 *  sh_hi, sh_lo [4][n_knots-1][4] coefficients of f_phi, f_r, Phi_phi, Phi_r (sh_lo may be NULL)
 *  am_hi, am_lo [n_modes][2][n_knots-1][4] coefficients of Re A, Im A (am_lo may be NULL)
 *  freq         [n_freq] sorted ascending, >= 0
 *  hplus,hcross [n_freq][2] (re, im), fully overwritten
 *  n_evals      out: number of accumulated (voice, sign, root, bin) terms (P9)
 *  nterms       optional [n_freq] int32: terms accumulated into each bin
 *  ambiguous    optional [n_freq] uint8: 1 if the bin's membership hinges on rounding (R8)
 *  max_roots    optional out: max over (voice, sign, bin) of the number of roots found
 *  n_threads    OpenMP threads over disjoint bin ranges (<=0: all) */
int fdemri_oracle_sum(int n_modes, const int32_t* lmn, int n_knots, const double* t,
                      const double* fphi_k, const double* fr_k,
                      const double* sh_hi, const double* sh_lo,
                      const double* am_hi, const double* am_lo,
                      int64_t n_freq, const double* freq, double theta, double phi,
                      double* hplus, double* hcross,
                      int64_t* n_evals, int32_t* nterms, uint8_t* ambiguous, int32_t* max_roots,
                      int n_threads);

/* Build (long double) + sum in one call: the level-C oracle.
 *  f_phi, f_r, Phi_phi, Phi_r [n_knots]; amp [n_modes][n_knots][2] (re, im). */
int fdemri_oracle_waveform(int n_modes, const int32_t* lmn, int n_knots, const double* t,
                           const double* f_phi, const double* f_r, const double* Phi_phi, const double* Phi_r,
                           const double* amp,
                           int64_t n_freq, const double* freq, double theta, double phi,
                           double* hplus, double* hcross,
                           int64_t* n_evals, int32_t* nterms, uint8_t* ambiguous, int32_t* max_roots,
                           int n_threads);

/* The same for general voices (l, m, k, n) of Eq. 1 (L64): F = m f_phi + k f_theta + n f_r, phase likewise, partner
 * (l,-m,-k,-n) implied for m > 0 with amplitude (-1)^(l+k) conj A; spherical harmonics stand in for the spheroidal ones
 * (L66: "Future work will describe how we handle this complication"; R16).  lmkn [n_modes][4]. */
int fdemri_oracle_waveform_kerr(int n_modes, const int32_t* lmkn, int n_knots, const double* t,
                                const double* f_phi, const double* f_theta, const double* f_r,
                                const double* Phi_phi, const double* Phi_theta, const double* Phi_r,
                                const double* amp,
                                int64_t n_freq, const double* freq, double theta, double phi,
                                double* hplus, double* hcross,
                                int64_t* n_evals, int32_t* nterms, uint8_t* ambiguous, int32_t* max_roots,
                                int n_threads);

/* Eq. 12 (L134-141) on a frequency grid, both polarisations: <a|b> = sum_k w_k [a+ conj b+ + ax conj bx],
 * w_k = 4 df / S_n(f_k) (NULL: w = 1).  hplus, hcross, dplus, dcross: [n_freq][2].  out = {<h|h>, Re<d|h>, Im<d|h>}.
 * hann != 0: h is first convolved with the DFT of the Hann window, h_k/2 - h_{k-1}/4 - h_{k+1}/4 (L145). */
int fdemri_oracle_inner(int64_t n_freq, const double* w, const double* hplus, const double* hcross,
                        const double* dplus, const double* dcross, int hann, double* out);

/* The time-domain voice sum the stationary-phase sum approximates (Eq. 1 / Eq. 2): on the uniform
 * time grid t_j = t0 + j dt, j = 0..n_samples-1,
 *     h(t) = h+ - i hx = sum over the list voices of  A_v(t) Y_lm e^{-i Phi_v(t)}
 *                        + for m > 0 the implied partner (l,-m,-k,-n):  (-1)^(l+k) conj(A_v(t)) Y_l,-m e^{+i Phi_v(t)},
 * with the not-a-knot splines of Phi_phi, Phi_r (, Phi_theta), Re A_v, Im A_v evaluated in long double, Phi_v formed
 * coefficient-wise (L103).  Samples outside [t_0, t_{N-1}) are 0 (R14).  lmkn [n_modes][4] (l, m, k, n); Phi_theta may be
 * NULL when every k is 0.  hplus, hcross: [n_samples] real. */
int fdemri_oracle_td(int n_modes, const int32_t* lmkn, int n_knots, const double* t,
                     const double* Phi_phi, const double* Phi_theta, const double* Phi_r, const double* amp,
                     int64_t n_samples, double t0, double dt, double theta, double phi,
                     double* hplus, double* hcross, int n_threads);

int fdemri_oracle_num_threads(void);
/* Test switch for pin P7: list voices stand for themselves only (m of either sign, no implied partner). */
void fdemri_oracle_set_explicit(int on);

#ifdef __cplusplus
}
#endif
#endif
