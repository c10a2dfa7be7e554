// fdemri_oracle.cpp -- CPU oracle for the FD EMRI harmonic sum (arXiv:2307.12585).
//
// TEST INFRASTRUCTURE ONLY (see fdemri_oracle.h).  Shares no code with the CUDA library.
// Compile: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC
// (-ffp-contract=off: the knot values F_k of R6 must be the plainly rounded doubles.)
//
// Everything is long double (x87, 64-bit mantissa) applied to the given double inputs.
#include "fdemri_oracle.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;
typedef std::complex<ld> cld;

static const ld PI_L = 3.141592653589793238462643383279502884L;
static const ld TWO_PI_L = 2.0L * PI_L;

// ---------------------------------------------------------------------------------------------
// O1. Not-a-knot cubic spline ("not-a-knot cubic spline"; L105 coefficients determined
// along the sparse trajectory).  Unknowns: second derivatives M_k at the knots.
//   interior rows k=1..N-2:  h_{k-1} M_{k-1} + 2(h_{k-1}+h_k) M_k + h_k M_{k+1}
//                              = 6[(y_{k+1}-y_k)/h_k - (y_k-y_{k-1})/h_{k-1}]
//   first row (third derivative continuous at t_1):   h_1 M_0 - (h_0+h_1) M_1 + h_0 M_2 = 0
//   last row (mirror, at t_{N-2}):  h_{N-2} M_{N-3} - (h_{N-3}+h_{N-2}) M_{N-2} + h_{N-3} M_{N-1} = 0
// Solved as a dense N x N system by Gaussian elimination with partial pivoting (factor once per knot
// set, back-substitute per component).  Segment k, tau = t - t_k:
//   a = y_k,  b = (y_{k+1}-y_k)/h_k - h_k (2 M_k + M_{k+1})/6,  c = M_k/2,  d = (M_{k+1}-M_k)/(6 h_k).
// ---------------------------------------------------------------------------------------------
struct KnotSystem {
    int N;
    std::vector<ld> h;     // N-1
    std::vector<ld> lu;    // N*N, row-major, LU in place
    std::vector<int> piv;  // row permutation
    explicit KnotSystem(int n, const double* t) : N(n), h(n - 1), lu((size_t)n * n, 0.0L), piv(n) {
        for (int k = 0; k < N - 1; ++k) h[k] = (ld)t[k + 1] - (ld)t[k];
        auto Mx = [&](int r, int c) -> ld& { return lu[(size_t)r * N + c]; };
        Mx(0, 0) = h[1];
        Mx(0, 1) = -(h[0] + h[1]);
        Mx(0, 2) = h[0];
        for (int k = 1; k <= N - 2; ++k) {
            Mx(k, k - 1) = h[k - 1];
            Mx(k, k) = 2.0L * (h[k - 1] + h[k]);
            Mx(k, k + 1) = h[k];
        }
        Mx(N - 1, N - 3) = h[N - 2];
        Mx(N - 1, N - 2) = -(h[N - 3] + h[N - 2]);
        Mx(N - 1, N - 1) = h[N - 3];
        for (int i = 0; i < N; ++i) piv[i] = i;
        for (int c = 0; c < N; ++c) {
            int best = c;
            for (int r = c + 1; r < N; ++r)
                if (fabsl(Mx(r, c)) > fabsl(Mx(best, c))) best = r;
            if (best != c) {
                for (int j = 0; j < N; ++j) std::swap(Mx(c, j), Mx(best, j));
                std::swap(piv[c], piv[best]);
            }
            for (int r = c + 1; r < N; ++r) {
                ld f = Mx(r, c) / Mx(c, c);
                Mx(r, c) = f;
                if (f != 0.0L)
                    for (int j = c + 1; j < N; ++j) Mx(r, j) -= f * Mx(c, j);
            }
        }
    }
    // coef: [N-1][4]
    void solve(const double* y, ld* coef) const {
        std::vector<ld> rhs(N, 0.0L), x(N);
        for (int k = 1; k <= N - 2; ++k)
            rhs[k] = 6.0L * (((ld)y[k + 1] - (ld)y[k]) / h[k] - ((ld)y[k] - (ld)y[k - 1]) / h[k - 1]);
        for (int i = 0; i < N; ++i) x[i] = rhs[piv[i]];
        for (int i = 0; i < N; ++i)
            for (int j = 0; j < i; ++j) x[i] -= lu[(size_t)i * N + j] * x[j];
        for (int i = N - 1; i >= 0; --i) {
            for (int j = i + 1; j < N; ++j) x[i] -= lu[(size_t)i * N + j] * x[j];
            x[i] /= lu[(size_t)i * N + i];
        }
        for (int k = 0; k < N - 1; ++k) {
            coef[4 * k + 0] = (ld)y[k];
            coef[4 * k + 1] = ((ld)y[k + 1] - (ld)y[k]) / h[k] - h[k] * (2.0L * x[k] + x[k + 1]) / 6.0L;
            coef[4 * k + 2] = x[k] / 2.0L;
            coef[4 * k + 3] = (x[k + 1] - x[k]) / (6.0L * h[k]);
        }
    }
};

static bool knots_ok(int n_knots, const double* t) {
    if (n_knots < 4 || !t) return false;
    for (int k = 0; k + 1 < n_knots; ++k)
        if (!(t[k + 1] > t[k])) return false;
    return true;
}

extern "C" int fdemri_oracle_build_splines(int n_knots, const double* t, int n_comp, const double* y,
                                           double* coef_hi, double* coef_lo) {
    if (!knots_ok(n_knots, t) || n_comp < 0 || !y || !coef_hi) return 1;
    KnotSystem ks(n_knots, t);
    size_t per = (size_t)(n_knots - 1) * 4;
    std::vector<ld> c(per);
    for (int q = 0; q < n_comp; ++q) {
        ks.solve(y + (size_t)q * n_knots, c.data());
        for (size_t i = 0; i < per; ++i) {
            double hi = (double)c[i];
            coef_hi[q * per + i] = hi;
            if (coef_lo) coef_lo[q * per + i] = (double)(c[i] - (ld)hi);
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Spin-weight s = -2 spherical harmonics (L66: for Schwarzschild the spheroidal harmonics are the
// spin-weighted spherical harmonics).  Goldberg et al. (1967) sum, written with sin/cos of theta/2:
//  sY_lm = (-1)^m sqrt[(l+m)!(l-m)!(2l+1) / (4 pi (l+s)!(l-s)!)] e^{i m phi}
//          * sum_r C(l-s, r) C(l+s, r+s-m) (-1)^{l-r-s} sin^{2l-2r-s+m}(theta/2) cos^{2r+s-m}(theta/2)
// ---------------------------------------------------------------------------------------------
static ld factl(int n) {
    ld f = 1.0L;
    for (int i = 2; i <= n; ++i) f *= (ld)i;
    return f;
}
static ld binoml(int n, int k) {
    if (k < 0 || k > n) return 0.0L;
    return factl(n) / (factl(k) * factl(n - k));
}
static cld ylm_m2(int l, int m, ld theta, ld phi) {
    const int s = -2;
    if (l < 2 || m > l || m < -l) return cld(0.0L, 0.0L);
    ld sh = sinl(theta / 2.0L), ch = cosl(theta / 2.0L);
    ld pref = sqrtl(factl(l + m) * factl(l - m) * (2.0L * l + 1.0L) / (4.0L * PI_L * factl(l + s) * factl(l - s)));
    if (m & 1) pref = -pref;
    ld sum = 0.0L;
    for (int r = 0; r <= l - s; ++r) {
        int ec = 2 * r + s - m;           // power of cos(theta/2)
        int es = 2 * l - 2 * r - s + m;   // power of sin(theta/2)
        ld bc = binoml(l - s, r) * binoml(l + s, r + s - m);
        if (bc == 0.0L) continue;
        ld term = bc * powl(sh, (ld)es) * powl(ch, (ld)ec);
        if ((l - r - s) & 1) term = -term;
        sum += term;
    }
    return pref * sum * cld(cosl((ld)m * phi), sinl((ld)m * phi));
}

extern "C" int fdemri_oracle_ylm(int l, int m, double theta, double phi, double* re, double* im) {
    if (l < 2 || m > l || m < -l || !re || !im) return 1;
    cld y = ylm_m2(l, m, (ld)theta, (ld)phi);
    *re = (double)y.real();
    *im = (double)y.imag();
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O3. Per-root factor of Eq. 9 (L107-119) as read in DESIGN.md R3/R4:
//   X = 2 pi Fdot^3 / (3 Fddot^2),
//   g(X) = sqrt(pi|X|/2) e^{i pi/6} e^{-i|X|} H^(1)_{1/3}(|X|)  (X>0),  conj for X<0,
//   factor = g(X)/sqrt|Fdot|.   g -> e^{-+ i pi/4} (standard SPA, L119) as |X| -> inf.
// Regular form for Fdot -> 0:  g/sqrt|Fdot| = e^{-iX} pi (pi|Fddot|)^{-1/3} [Ai(-y) -+ i Bi(-y)],
//   y = (3|X|/2)^{2/3}, upper sign for Fdot>0.
// ---------------------------------------------------------------------------------------------
static cld g_asymptotic(ld ax) {   // ax = |X| > 30;  g = e^{-i pi/4} sum_k i^k a_k / ax^k, K = 16
    ld ak = 1.0L, pw = 1.0L, re = 1.0L, im = 0.0L;
    for (int k = 1; k <= 16; ++k) {
        ld odd = (ld)(2 * k - 1);
        ak *= (4.0L / 9.0L - odd * odd) / ((ld)k * 8.0L);
        pw /= ax;
        ld term = ak * pw;
        switch (k & 3) {
            case 0: re += term; break;
            case 1: im += term; break;
            case 2: re -= term; break;
            case 3: im -= term; break;
        }
    }
    const ld r = sqrtl(0.5L);
    return cld(re, im) * cld(r, -r);
}
static cld g_bessel(ld ax) {   // 1e-8 <= ax <= 30
    const ld nu = 1.0L / 3.0L;
    ld J = std::cyl_bessel_j(nu, ax);
    ld Y = std::cyl_neumann(nu, ax);
    cld H(J, Y);
    ld amp = sqrtl(PI_L * ax / 2.0L);
    ld ph = PI_L / 6.0L - ax;
    return amp * cld(cosl(ph), sinl(ph)) * H;
}
static cld g_of_X(ld X) {
    ld ax = fabsl(X);
    cld g;
    if (ax > 30.0L) g = g_asymptotic(ax);
    else if (ax >= 1e-8L) g = g_bessel(ax);
    else {
        // tiny |X|: g = sqrt|Fdot| * (regular form); with y = (3ax/2)^{2/3}:  sqrt|Fdot| (pi|Fddot|)^{-1/3}
        // = (y/pi^2)^{1/4} ... written directly: g = e^{-i ax} pi^{1/2} y^{1/4} [Ai(-y) - i Bi(-y)]
        ld y = powl(1.5L * ax, 2.0L / 3.0L);
        const ld ai0 = 0.355028053887817239260063186004183177L, aip0 = -0.258819403792806798405183560189203963L;
        const ld bi0 = 0.614926627446000735150922369093613554L, bip0 = 0.448288357353826357914823710398828140L;
        ld z = -y;
        ld f = 1.0L + z * z * z / 6.0L, gg = z + z * z * z * z / 12.0L;
        ld Ai = ai0 * f + aip0 * gg, Bi = bi0 * f + bip0 * gg;
        g = cld(cosl(ax), -sinl(ax)) * sqrtl(PI_L) * powl(y, 0.25L) * cld(Ai, -Bi);
    }
    return X >= 0.0L ? g : std::conj(g);
}

extern "C" int fdemri_oracle_g(double X, double* re, double* im) {
    if (!re || !im || !(X == X)) return 1;
    cld g = g_of_X((ld)X);
    *re = (double)g.real();
    *im = (double)g.imag();
    return 0;
}

// returns false when there is no term (R10: Fdot = Fddot = 0)
static bool g_over_sqrt(ld Fd, ld Fdd, cld* out) {
    if (Fdd == 0.0L) {
        if (Fd == 0.0L) return false;
        const ld r = sqrtl(0.5L);
        *out = cld(r, Fd > 0 ? -r : r) / sqrtl(fabsl(Fd));   // standard SPA, e^{-+ i pi/4}/sqrt|Fdot|
        return true;
    }
    ld X = TWO_PI_L * Fd * Fd * Fd / (3.0L * Fdd * Fdd);
    ld ax = fabsl(X);
    if (ax >= 1e-8L) {
        *out = g_of_X(X) / sqrtl(fabsl(Fd));
        return true;
    }
    // Airy regular form, valid down to Fdot = 0
    ld y = powl(1.5L * ax, 2.0L / 3.0L);
    const ld ai0 = 0.355028053887817239260063186004183177L, aip0 = -0.258819403792806798405183560189203963L;
    const ld bi0 = 0.614926627446000735150922369093613554L, bip0 = 0.448288357353826357914823710398828140L;
    ld z = -y;
    ld f = 1.0L + z * z * z / 6.0L, gg = z + z * z * z * z / 12.0L;
    ld Ai = ai0 * f + aip0 * gg, Bi = bi0 * f + bip0 * gg;
    cld v = cld(cosl(ax), -sinl(ax)) * PI_L * powl(PI_L * fabsl(Fdd), -1.0L / 3.0L) * cld(Ai, -Bi);
    *out = (Fd >= 0.0L) ? v : std::conj(v);
    return true;
}

extern "C" int fdemri_oracle_g_over_sqrt(double Fdot, double Fddot, double* re, double* im) {
    cld v;
    if (!g_over_sqrt((ld)Fdot, (ld)Fddot, &v)) return 1;
    *re = (double)v.real();
    *im = (double)v.imag();
    return 0;
}

// ---------------------------------------------------------------------------------------------
// O2. The sum.
// ---------------------------------------------------------------------------------------------
struct Piece {            // one monotone piece of one segment of one voice (R6, R7)
    int seg;
    ld ta, tb;            // tau range inside the segment
    double Va, Vb;        // F at the ends: knot values (doubles, R6) or F_e (R7)
    bool a_incl, b_incl;  // membership includes the value Va / Vb
    bool a_ext, b_ext;    // end is an interior extremum (for R8 bookkeeping)
};

struct Voice {
    int l, m, n, k;                    // k: polar harmonic of the general voice (l, m, k, n) of Eq. 1; 0 in Schwarzschild
    std::vector<ld> cF, cP, cRe, cIm;  // [N-1][4] coefficient-wise voice splines (L103)
    std::vector<Piece> pieces;
    cld Wp, Wx;
};

static inline ld horner3(const ld* c, ld x) { return c[0] + x * (c[1] + x * (c[2] + x * c[3])); }

static inline double ulp_of(double v) {
    double a = fabs(v);
    return nextafter(a, INFINITY) - a;
}

// root of F(tau) = x on a monotone piece, safeguarded Newton / bisection in long double
static ld solve_piece(const ld* c, ld x, ld ta, ld tb) {
    ld Ga = horner3(c, ta) - x, Gb = horner3(c, tb) - x;
    if (Ga == 0.0L) return ta;
    if (Gb == 0.0L) return tb;
    if ((Ga > 0) == (Gb > 0)) return fabsl(Ga) < fabsl(Gb) ? ta : tb;   // rounding at an end: clamp (R6)
    ld lo = ta, hi = tb;            // G(lo) < 0 < G(hi) after orientation
    if (Ga > 0) { lo = tb; hi = ta; }
    ld tau = 0.5L * (ta + tb), dold = fabsl(tb - ta), d = dold;
    ld G = horner3(c, tau) - x, dG = c[1] + tau * (2.0L * c[2] + tau * 3.0L * c[3]);
    for (int it = 0; it < 300; ++it) {
        bool newton_out = ((tau - hi) * dG - G) * ((tau - lo) * dG - G) > 0.0L;
        if (newton_out || fabsl(2.0L * G) > fabsl(dold * dG)) {
            dold = d;
            d = 0.5L * (hi - lo);
            tau = lo + d;
            if (lo == tau) return tau;
        } else {
            dold = d;
            d = G / dG;
            ld prev = tau;
            tau -= d;
            if (prev == tau) return tau;
        }
        if (fabsl(d) < 2e-19L * fabsl(tb - ta)) return tau;
        G = horner3(c, tau) - x;
        dG = c[1] + tau * (2.0L * c[2] + tau * 3.0L * c[3]);
        if (G < 0) lo = tau; else hi = tau;
    }
    return tau;
}

// Interior extrema of the segment cubic F(tau) = c0 + c1 tau + c2 tau^2 + c3 tau^3 on (0, h): the points where
// F'(tau) = c1 + 2 c2 tau + 3 c3 tau^2 changes sign (R7: "interior extremum tau_e from F'(tau) = 0").
// F' is a parabola: monotone on either side of its vertex, so every sign change of F' on [0, h] is bracketed by
// consecutive points of {0, vertex (if inside), h} and found by bisection to the last bit of long double.
// (A double root of F' -- an inflection with a horizontal tangent -- is not a sign change and gives no extremum.)
static void interior_extrema(const ld* c, ld h, ld* ext, int* ne) {
    auto dF = [&](ld tau) { return c[1] + tau * (2.0L * c[2] + tau * 3.0L * c[3]); };
    ld pts[3]; int np = 0;
    pts[np++] = 0.0L;
    if (c[3] != 0.0L) {
        const ld tv = -c[2] / (3.0L * c[3]);              // vertex of the parabola F'
        if (tv > 0.0L && tv < h) pts[np++] = tv;
    }
    pts[np++] = h;
    *ne = 0;
    for (int j = 0; j + 1 < np; ++j) {
        ld a = pts[j], b = pts[j + 1];
        ld fa = dF(a), fb = dF(b);
        if (!((fa < 0.0L && fb > 0.0L) || (fa > 0.0L && fb < 0.0L))) continue;   // no strict sign change
        for (;;) {
            const ld mid = a + 0.5L * (b - a);
            if (!(mid > a && mid < b)) break;             // the bracket has collapsed to neighbouring numbers
            const ld fm = dF(mid);
            if (fm == 0.0L) { a = b = mid; break; }
            if ((fm < 0.0L) == (fa < 0.0L)) { a = mid; fa = fm; } else { b = mid; }
        }
        const ld r = a + 0.5L * (b - a);
        if (r > 0.0L && r < h && *ne < 2) ext[(*ne)++] = r;
    }
}

// Test switch (pin P7): when set, every list voice (any sign of m) stands for itself only -- no implied
// (l,-m,-n) partner -- and contributes S(f) Y_lm to h~(f), i.e. W+ = Y/2, Wx = iY/2.
static int g_explicit_voices = 0;
extern "C" void fdemri_oracle_set_explicit(int on) { g_explicit_voices = on; }

/* Eq. 12, both polarisations, as the plain sum it is on a frequency grid:
 *   <a|b> = sum_k w_k [ a+(f_k) conj b+(f_k) + ax(f_k) conj bx(f_k) ],   w_k = 4 df / S_n(f_k)  (w = 1 if NULL).
 * The paper's inner product is the real part; the imaginary part is returned as well.  long double sums in index
 * order.  out = {<h|h>, Re<d|h>, Im<d|h>};  d may be NULL (then only out[0] is set).
 * hann != 0: h is first replaced by its convolution with the DFT of the Hann window (L145):
 *   h_k <- h_k/2 - h_{k-1}/4 - h_{k+1}/4,  bins outside the grid counting as zero. */
extern "C" int fdemri_oracle_inner(int64_t n_freq, const double* w, const double* hplus, const double* hcross,
                                   const double* dplus, const double* dcross, int hann, double* out) {
    if (n_freq < 0 || !hplus || !hcross || !out) return 1;
    long double hh = 0.0L, dr = 0.0L, di = 0.0L;
    auto at = [&](const double* h, int64_t k, int c) -> long double {
        return (k < 0 || k >= n_freq) ? 0.0L : (long double)h[2 * k + c];
    };
    auto val = [&](const double* h, int64_t k, int c) -> long double {
        if (!hann) return at(h, k, c);
        return 0.5L * at(h, k, c) - 0.25L * at(h, k - 1, c) - 0.25L * at(h, k + 1, c);
    };
    for (int64_t k = 0; k < n_freq; ++k) {
        const long double wk = w ? (long double)w[k] : 1.0L;
        const long double pr = val(hplus, k, 0), pi = val(hplus, k, 1), xr = val(hcross, k, 0), xi = val(hcross, k, 1);
        hh += wk * (pr * pr + pi * pi + xr * xr + xi * xi);
        if (dplus && dcross) {
            const long double ar = dplus[2 * k], ai = dplus[2 * k + 1], br = dcross[2 * k], bi = dcross[2 * k + 1];
            /* d conj(h) = (ar + i ai)(pr - i pi) */
            dr += wk * (ar * pr + ai * pi + br * xr + bi * xi);
            di += wk * (ai * pr - ar * pi + bi * xr - br * xi);
        }
    }
    out[0] = (double)hh; out[1] = (double)dr; out[2] = (double)di;
    return 0;
}

// kk, fth_k NULL: Schwarzschild voices (l, m, n).  Otherwise kk[v] is the polar harmonic k of voice v (Eq. 1:
// phase m Phi_phi + k Phi_theta + n Phi_r), fth_k the knot values of f_theta, and sh holds six splines.
static int sum_impl(int n_modes, const int32_t* lmn, const int32_t* kk, int N, const double* t,
                    const double* fphi_k, const double* fth_k, const double* fr_k,
                    const ld* sh,      // [4][N-1][4]: f_phi, f_r, Phi_phi, Phi_r  (+ f_theta, Phi_theta: [6][N-1][4])
                    const ld* am,      // [n_modes][2][N-1][4]
                    int64_t n_freq, const double* freq, double theta, double phi,
                    double* hplus, double* hcross,
                    int64_t* n_evals_out, int32_t* nterms, uint8_t* ambiguous, int32_t* max_roots_out,
                    int n_threads) {
    if (n_modes < 0 || !lmn || !knots_ok(N, t) || n_freq < 0 || !freq || !hplus || !hcross) return 1;
    for (int64_t i = 0; i < n_freq; ++i) {
        if (!(freq[i] >= 0.0)) return 1;
        if (i && !(freq[i] > freq[i - 1])) return 1;
    }
    const int S = N - 1;
    const size_t per = (size_t)S * 4;
    std::vector<Voice> voices(n_modes);
    for (int v = 0; v < n_modes; ++v) {
        Voice& V = voices[v];
        V.l = lmn[3 * v]; V.m = lmn[3 * v + 1]; V.n = lmn[3 * v + 2];
        V.k = kk ? kk[v] : 0;
        if (V.l < 2 || (V.m < 0 && !g_explicit_voices) || V.m > V.l || V.m < -V.l) return 1;
        V.cF.resize(per); V.cP.resize(per); V.cRe.resize(per); V.cIm.resize(per);
        for (size_t i = 0; i < per; ++i) {
            // L103: A..D "given by the sum of the spline coefficients ... multiplied by their mode number"
            V.cF[i] = (ld)V.m * sh[0 * per + i] + (ld)V.n * sh[1 * per + i];
            V.cP[i] = (ld)V.m * sh[2 * per + i] + (ld)V.n * sh[3 * per + i];
            if (kk) {
                V.cF[i] += (ld)V.k * sh[4 * per + i];
                V.cP[i] += (ld)V.k * sh[5 * per + i];
            }
            V.cRe[i] = am[((size_t)v * 2 + 0) * per + i];
            V.cIm[i] = am[((size_t)v * 2 + 1) * per + i];
        }
        // O2 weights
        cld Y = ylm_m2(V.l, V.m, theta, phi);
        if (V.m > 0 && !g_explicit_voices) {
            cld Ym = std::conj(ylm_m2(V.l, -V.m, theta, phi));
            ld sg = ((V.l + V.k) & 1) ? -1.0L : 1.0L;     // (-1)^(l+k): partner (l,-m,-k,-n), R16
            V.Wp = 0.5L * (Y + sg * Ym);
            V.Wx = cld(0.0L, 0.5L) * (Y - sg * Ym);
        } else {
            V.Wp = 0.5L * Y;
            V.Wx = cld(0.0L, 0.5L) * Y;
        }
        // knot values of F_v as plainly rounded doubles (R6)
        std::vector<double> Fk(N);
        for (int k = 0; k < N; ++k) {
            double pm = (double)V.m * fphi_k[k];
            double pn = (double)V.n * fr_k[k];
            if (kk) {                              // Eq. 1's order: (m f_phi + k f_theta) + n f_r, each step rounded
                double pk = (double)V.k * fth_k[k];
                pm = pm + pk;
            }
            Fk[k] = pm + pn;
        }
        // pieces: split every segment at the interior extrema of its cubic (R5, R7)
        for (int k = 0; k < S; ++k) {
            const ld* c = &V.cF[4 * k];
            ld h = (ld)t[k + 1] - (ld)t[k];
            ld ext[2]; int ne = 0;
            interior_extrema(c, h, ext, &ne);
            ld brk[4]; double val[4]; int nb = 0;
            brk[nb] = 0.0L; val[nb++] = Fk[k];
            for (int e = 0; e < ne; ++e) { brk[nb] = ext[e]; val[nb++] = (double)horner3(c, ext[e]); }
            brk[nb] = h; val[nb++] = Fk[k + 1];
            for (int j = 0; j + 1 < nb; ++j) {
                Piece P;
                P.seg = k; P.ta = brk[j]; P.tb = brk[j + 1]; P.Va = val[j]; P.Vb = val[j + 1];
                P.a_ext = (j > 0); P.b_ext = (j + 2 < nb);
                P.a_incl = !P.a_ext;     // starts at the knot: included; starts at an extremum: excluded
                P.b_incl = P.b_ext;      // ends at an extremum: included; ends at the next knot: excluded
                if (P.Va != P.Vb) V.pieces.push_back(P);
            }
        }
    }

    std::vector<ld> acc((size_t)n_freq * 4, 0.0L);
    if (nterms) std::memset(nterms, 0, sizeof(int32_t) * (size_t)n_freq);
    if (ambiguous) std::memset(ambiguous, 0, (size_t)n_freq);
    int64_t n_evals = 0;
    int max_roots = 0;
#ifdef _OPENMP
    omp_set_num_threads(n_threads > 0 ? n_threads : omp_get_num_procs());
    const int n_thr = omp_get_max_threads();
#else
    const int n_thr = 1;
#endif
    // disjoint bin ranges, one at a time per thread: every bin is summed in voice order (deterministic)
    const int64_t CH = std::max<int64_t>(512, std::min<int64_t>(16384, n_freq / (16 * (int64_t)n_thr) + 1));
    const int64_t n_chunks = (n_freq + CH - 1) / CH;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : n_evals) reduction(max : max_roots)
    for (int64_t ch = 0; ch < n_chunks; ++ch) {
        const int64_t c0 = ch * CH, c1 = std::min(n_freq, c0 + CH);
        const double* fb = freq + c0;
        const double* fe = freq + c1;
        if (c1 <= c0) continue;
        // roots found per (voice, sign, bin): stamp = id of the (voice, sign) that last touched the bin
        std::vector<int> stamp((size_t)(c1 - c0), -1), cnt((size_t)(c1 - c0), 0);
        const double ch_lo = fb[0] * (1.0 - 1e-13), ch_hi = fe[-1] * (1.0 + 1e-13);
        for (int v = 0; v < n_modes; ++v) {
            const Voice& V = voices[v];
            for (int sgn = +1; sgn >= -1; sgn -= 2) {
                const int vs_id = 2 * v + (sgn < 0);
                for (const Piece& P : V.pieces) {
                    // members: s*f between Va and Vb (inclusive/exclusive per R6/R7), f > 0
                    double lo_v = std::min(P.Va, P.Vb), hi_v = std::max(P.Va, P.Vb);
                    bool lo_incl = (P.Va < P.Vb) ? P.a_incl : P.b_incl;
                    bool hi_incl = (P.Va < P.Vb) ? P.b_incl : P.a_incl;
                    // in terms of f = s*x:  s=+1: f in [lo_v, hi_v];  s=-1: f in [-hi_v, -lo_v]
                    double flo = sgn > 0 ? lo_v : -hi_v, fhi = sgn > 0 ? hi_v : -lo_v;
                    bool flo_incl = sgn > 0 ? lo_incl : hi_incl, fhi_incl = sgn > 0 ? hi_incl : lo_incl;
                    if (fhi < ch_lo || flo > ch_hi) continue;      // piece does not reach this bin range
                    const double* pb = flo_incl ? std::lower_bound(fb, fe, flo) : std::upper_bound(fb, fe, flo);
                    const double* pe = fhi_incl ? std::upper_bound(fb, fe, fhi) : std::lower_bound(fb, fe, fhi);
                    if (ambiguous) {
                        // R8: bins within a few ulp of an extremum value F_e -- the only boundary value that an
                        // independent implementation computes itself (knot values are the same doubles everywhere,
                        // so comparisons against them are exact and never ambiguous)
                        bool lo_ext = (P.Va < P.Vb) ? P.a_ext : P.b_ext, hi_ext = (P.Va < P.Vb) ? P.b_ext : P.a_ext;
                        bool flo_ext = sgn > 0 ? lo_ext : hi_ext, fhi_ext = sgn > 0 ? hi_ext : lo_ext;
                        if (flo_ext)
                            for (const double* q = pb - 1; q <= pb; ++q)
                                if (q >= fb && q < fe && fabs(*q - flo) <= 16.0 * ulp_of(flo) && *q > 0.0) ambiguous[q - freq] = 1;
                        if (fhi_ext)
                            for (const double* q = pe - 1; q <= pe; ++q)
                                if (q >= fb && q < fe && fabs(*q - fhi) <= 16.0 * ulp_of(fhi) && *q > 0.0) ambiguous[q - freq] = 1;
                    }
                    const ld* cF = &V.cF[4 * P.seg];
                    const ld* cP = &V.cP[4 * P.seg];
                    const ld* cR = &V.cRe[4 * P.seg];
                    const ld* cI = &V.cIm[4 * P.seg];
                    const ld tk = (ld)t[P.seg];
                    for (const double* q = pb; q < pe; ++q) {
                        const double f = *q;
                        if (!(f > 0.0)) continue;                      // R13: bin f = 0 -> 0
                        const ld x = (ld)sgn * (ld)f;                  // s*f
                        ld tau = solve_piece(cF, x, P.ta, P.tb);       // Eq. 6 inverted (L105)
                        ld Fd = cF[1] + tau * (2.0L * cF[2] + tau * 3.0L * cF[3]);   // L107: from the F spline
                        ld Fdd = 2.0L * cF[2] + 6.0L * cF[3] * tau;
                        cld gf;
                        if (!g_over_sqrt(Fd, Fdd, &gf)) continue;      // R10
                        cld A(horner3(cR, tau), horner3(cI, tau));
                        // phase psi = 2 pi (s f) t* - Phi_v(t*), t* = t_k + tau, kept in cycles (R9):
                        //   (s f) t_k exactly as p + e (fma), reduced mod 1
                        ld p = x * tk;
                        ld e = fmal(x, tk, -p);
                        ld cyc = (p - rintl(p)) + e;
                        cyc += x * tau;
                        ld Phi = horner3(cP, tau);
                        ld pc = Phi / TWO_PI_L;
                        cyc -= (pc - rintl(pc));
                        cyc -= rintl(cyc);
                        ld ang = TWO_PI_L * cyc;
                        cld Sterm = A * gf * cld(cosl(ang), sinl(ang));
                        cld tp = Sterm * V.Wp, tx = Sterm * V.Wx;
                        if (sgn < 0) { tp = std::conj(tp); tx = std::conj(tx); }
                        ld* a = &acc[(size_t)(q - freq) * 4];
                        a[0] += tp.real(); a[1] += tp.imag(); a[2] += tx.real(); a[3] += tx.imag();
                        ++n_evals;
                        if (nterms) ++nterms[q - freq];
                        const size_t j = (size_t)(q - fb);
                        if (stamp[j] != vs_id) { stamp[j] = vs_id; cnt[j] = 0; }
                        max_roots = std::max(max_roots, ++cnt[j]);
                    }
                }
            }
        }
    }
    for (int64_t i = 0; i < n_freq; ++i) {
        hplus[2 * i] = (double)acc[4 * i];
        hplus[2 * i + 1] = (double)acc[4 * i + 1];
        hcross[2 * i] = (double)acc[4 * i + 2];
        hcross[2 * i + 1] = (double)acc[4 * i + 3];
    }
    if (n_evals_out) *n_evals_out = n_evals;
    if (max_roots_out) *max_roots_out = max_roots;
    return 0;
}

extern "C" int fdemri_oracle_sum(int n_modes, const int32_t* lmn, int n_knots, const double* t,
                                 const double* fphi_k, const double* fr_k,
                                 const double* sh_hi, const double* sh_lo,
                                 const double* am_hi, const double* am_lo,
                                 int64_t n_freq, const double* freq, double theta, double phi,
                                 double* hplus, double* hcross,
                                 int64_t* n_evals, int32_t* nterms, uint8_t* ambiguous, int32_t* max_roots,
                                 int n_threads) {
    if (!knots_ok(n_knots, t) || !sh_hi || !am_hi || !fphi_k || !fr_k || n_modes < 0) return 1;
    size_t per = (size_t)(n_knots - 1) * 4;
    std::vector<ld> sh(4 * per), am((size_t)n_modes * 2 * per);
    for (size_t i = 0; i < sh.size(); ++i) sh[i] = (ld)sh_hi[i] + (sh_lo ? (ld)sh_lo[i] : 0.0L);
    for (size_t i = 0; i < am.size(); ++i) am[i] = (ld)am_hi[i] + (am_lo ? (ld)am_lo[i] : 0.0L);
    return sum_impl(n_modes, lmn, NULL, n_knots, t, fphi_k, NULL, fr_k, sh.data(), am.data(), n_freq, freq, theta, phi,
                    hplus, hcross, n_evals, nterms, ambiguous, max_roots, n_threads);
}

extern "C" int fdemri_oracle_waveform(int n_modes, const int32_t* lmn, int n_knots, const double* t,
                                      const double* f_phi, const double* f_r, const double* Phi_phi,
                                      const double* Phi_r, const double* amp,
                                      int64_t n_freq, const double* freq, double theta, double phi,
                                      double* hplus, double* hcross,
                                      int64_t* n_evals, int32_t* nterms, uint8_t* ambiguous, int32_t* max_roots,
                                      int n_threads) {
    if (!knots_ok(n_knots, t) || !f_phi || !f_r || !Phi_phi || !Phi_r || !amp || n_modes < 0) return 1;
    const int N = n_knots;
    size_t per = (size_t)(N - 1) * 4;
    KnotSystem ks(N, t);
    std::vector<ld> sh(4 * per), am((size_t)n_modes * 2 * per);
    ks.solve(f_phi, &sh[0 * per]);
    ks.solve(f_r, &sh[1 * per]);
    ks.solve(Phi_phi, &sh[2 * per]);
    ks.solve(Phi_r, &sh[3 * per]);
    std::vector<double> y(N);
    for (int v = 0; v < n_modes; ++v)
        for (int c = 0; c < 2; ++c) {
            for (int k = 0; k < N; ++k) y[k] = amp[((size_t)v * N + k) * 2 + c];
            ks.solve(y.data(), &am[((size_t)v * 2 + c) * per]);
        }
    return sum_impl(n_modes, lmn, NULL, N, t, f_phi, NULL, f_r, sh.data(), am.data(), n_freq, freq, theta, phi,
                    hplus, hcross, n_evals, nterms, ambiguous, max_roots, n_threads);
}

extern "C" int fdemri_oracle_waveform_kerr(int n_modes, const int32_t* lmkn, int n_knots, const double* t,
                                           const double* f_phi, const double* f_theta, const double* f_r,
                                           const double* Phi_phi, const double* Phi_theta, const double* Phi_r,
                                           const double* amp,
                                           int64_t n_freq, const double* freq, double theta, double phi,
                                           double* hplus, double* hcross,
                                           int64_t* n_evals, int32_t* nterms, uint8_t* ambiguous, int32_t* max_roots,
                                           int n_threads) {
    if (!knots_ok(n_knots, t) || !lmkn || !f_phi || !f_theta || !f_r || !Phi_phi || !Phi_theta || !Phi_r || !amp ||
        n_modes < 0)
        return 1;
    const int N = n_knots;
    size_t per = (size_t)(N - 1) * 4;
    KnotSystem ks(N, t);
    std::vector<ld> sh(6 * per), am((size_t)n_modes * 2 * per);
    ks.solve(f_phi, &sh[0 * per]);
    ks.solve(f_r, &sh[1 * per]);
    ks.solve(Phi_phi, &sh[2 * per]);
    ks.solve(Phi_r, &sh[3 * per]);
    ks.solve(f_theta, &sh[4 * per]);
    ks.solve(Phi_theta, &sh[5 * per]);
    std::vector<double> y(N);
    for (int v = 0; v < n_modes; ++v)
        for (int c = 0; c < 2; ++c) {
            for (int k = 0; k < N; ++k) y[k] = amp[((size_t)v * N + k) * 2 + c];
            ks.solve(y.data(), &am[((size_t)v * 2 + c) * per]);
        }
    std::vector<int32_t> lmn((size_t)n_modes * 3), kk(n_modes);
    for (int v = 0; v < n_modes; ++v) {            // (l, m, k, n) in the order of Eq. 1's subscript
        lmn[3 * v] = lmkn[4 * v]; lmn[3 * v + 1] = lmkn[4 * v + 1]; lmn[3 * v + 2] = lmkn[4 * v + 3];
        kk[v] = lmkn[4 * v + 2];
    }
    return sum_impl(n_modes, lmn.data(), kk.data(), N, t, f_phi, f_theta, f_r, sh.data(), am.data(), n_freq, freq,
                    theta, phi, hplus, hcross, n_evals, nterms, ambiguous, max_roots, n_threads);
}

// Eq. 1 / Eq. 2 (L62-74): the time-domain voice sum, sample by sample, voice by voice.
extern "C" int fdemri_oracle_td(int n_modes, const int32_t* lmkn, int n_knots, const double* t,
                                const double* Phi_phi, const double* Phi_theta, const double* Phi_r, const double* amp,
                                int64_t n_samples, double t0, double dt, double theta, double phi,
                                double* hplus, double* hcross, int n_threads) {
    if (!knots_ok(n_knots, t) || !lmkn || !Phi_phi || !Phi_r || !amp || n_modes < 0 || n_samples < 0 || !hplus || !hcross)
        return 1;
    const int N = n_knots, S = N - 1;
    const size_t per = (size_t)S * 4;
    KnotSystem ks(N, t);
    std::vector<ld> sp(3 * per, 0.0L), am((size_t)n_modes * 2 * per);
    ks.solve(Phi_phi, &sp[0 * per]);
    ks.solve(Phi_r, &sp[1 * per]);
    if (Phi_theta) ks.solve(Phi_theta, &sp[2 * per]);
    std::vector<double> y(N);
    std::vector<cld> Yp(n_modes), Ym(n_modes);
    for (int v = 0; v < n_modes; ++v) {
        const int l = lmkn[4 * v], m = lmkn[4 * v + 1], k = lmkn[4 * v + 2];
        if (l < 2 || m < 0 || m > l || (k != 0 && !Phi_theta)) return 1;
        for (int c = 0; c < 2; ++c) {
            for (int q = 0; q < N; ++q) y[q] = amp[((size_t)v * N + q) * 2 + c];
            ks.solve(y.data(), &am[((size_t)v * 2 + c) * per]);
        }
        Yp[v] = ylm_m2(l, m, theta, phi);
        const ld sg = ((l + k) & 1) ? -1.0L : 1.0L;                      // (-1)^(l+k), R16
        Ym[v] = (m > 0) ? sg * ylm_m2(l, -m, theta, phi) : cld(0.0L, 0.0L);
    }
#ifdef _OPENMP
    omp_set_num_threads(n_threads > 0 ? n_threads : omp_get_num_procs());
#endif
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n_samples; ++j) {
        const double tj = t0 + (double)j * dt;                           // the sample time as a double (product, then sum)
        hplus[j] = 0.0; hcross[j] = 0.0;
        if (!(tj >= t[0]) || !(tj < t[N - 1])) continue;                 // R14
        int seg = (int)(std::upper_bound(t, t + N, tj) - t) - 1;
        seg = std::min(std::max(seg, 0), S - 1);
        const ld tau = (ld)tj - (ld)t[seg];
        cld h(0.0L, 0.0L);
        for (int v = 0; v < n_modes; ++v) {
            const int m = lmkn[4 * v + 1], k = lmkn[4 * v + 2], n = lmkn[4 * v + 3];
            ld cP[4];
            for (int q = 0; q < 4; ++q)                                  // L103: coefficient-wise
                cP[q] = (ld)m * sp[0 * per + 4 * seg + q] + (ld)n * sp[1 * per + 4 * seg + q] + (ld)k * sp[2 * per + 4 * seg + q];
            const ld Phi = horner3(cP, tau);
            ld cyc = Phi / TWO_PI_L;
            cyc -= rintl(cyc);
            const ld ang = TWO_PI_L * cyc;
            const cld A(horner3(&am[((size_t)v * 2 + 0) * per + 4 * seg], tau), horner3(&am[((size_t)v * 2 + 1) * per + 4 * seg], tau));
            const cld E(cosl(ang), -sinl(ang));                          // e^{-i Phi}
            h += A * Yp[v] * E;
            if (m > 0) h += std::conj(A) * Ym[v] * std::conj(E);
        }
        hplus[j] = (double)h.real();                                     // h = h+ - i hx (L64)
        hcross[j] = (double)(-h.imag());
    }
    return 0;
}

extern "C" int fdemri_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
