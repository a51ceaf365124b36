// =====================================================================================
//  picsarqed_oracle.cpp  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
//  A plain, slow, CPU-only restatement of what the PICSAR-QED method computes
//  (arXiv 2110.00256; cited below as PAPER.md:<line>).  It exists so that the CUDA
//  library in paper_2110_00256_b200/ can be checked element by element.  Only tests/,
//  __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
//  it.  It shares no code, header, table or constant generator with the CUDA path.
//
//  Two halves:
//   (I)  table definitions, evaluated by adaptive Gauss-Kronrod quadrature in
//        fp64: T(chi_gamma) eq.9, the Breit-Wheeler CDF eq.11, G(chi) eqs.16-17,
//        the photon-emission CDF eq.18.  K_nu and its tail integral are evaluated from
//        the integral representation K_nu(x) = int_0^inf exp(-x cosh t) cosh(nu t) dt
//        (DLMF 10.32.9), which is a *definition*, and is pinned in tests/ against
//        scipy's kve (AMOS), mpmath, K_{1/2} and Airy closed forms.
//   (II) the runtime algorithm, step by step in the paper's order: chi (eqs.2-3) in
//        __float128, the 1D log-log lookups (eqs.23, 27), the optical-depth update
//        (PAPER.md:195), the inverse-CDF events (eqs.24-26, 28-30), Philox4x32-10
//        uniforms, and the serial, index-ordered creation of secondaries.
//
//  Readings of garbled / silent passages are listed in DESIGN.md ("Readings").
//  Parity pins: every exported function below is pinned by tests/test_oracle_*.py;
//  the single exception is the QS draw below the first table column (r < P(xi_min)),
//  which the paper does not fix: "parity unpinned" for that branch only (R6).
//
//  Build: g++ -O2 -std=c++17 -fopenmp -fPIC -shared picsarqed_oracle.cpp -lquadmath
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double real;  // runtime half (II); chi itself is done in __float128
typedef double treal;      // table half (I): fp64 throughout

static const real PI_L = 3.14159265358979323846264338327950288L;

// -------------------------------------------------------------------------------------
//  Physical constants (CODATA 2018 exact/recommended values; eq.1 gives
//  only E_s ~ 1.32e18 V/m, which orc_schwinger_field() reproduces).
// -------------------------------------------------------------------------------------
static const real C_LIGHT = 299792458.0L;            // m/s
static const real H_PLANCK = 6.62607015e-34L;        // J s
static const real Q_ELEM = 1.602176634e-19L;            // C
static const real M_ELECTRON = 9.1093837015e-31L;           // kg
static const real ALPHA_F = 7.2973525693e-3L;        // fine-structure constant
static inline real hbar() { return H_PLANCK / (2 * PI_L); }
// alpha_f m_e c^2 / hbar  [1/s]: the prefactor of eq.8 and eq.15
static inline real rate_prefactor() { return ALPHA_F * M_ELECTRON * C_LIGHT * C_LIGHT / hbar(); }

// -------------------------------------------------------------------------------------
//  Adaptive 7-15 Gauss-Kronrod quadrature (nodes/weights: Piessens et al., QUADPACK).
//  orc_selftest_gk15() checks that the typed constants integrate x^k exactly, k <= 22.
// -------------------------------------------------------------------------------------
static const real XGK[8] = {
    0.991455371120812639206854697526329L, 0.949107912342758524526189684047851L,
    0.864864423359769072789712788640926L, 0.741531185599394439863864773280788L,
    0.586087235467691130294144838258730L, 0.405845151377397166906606412076961L,
    0.207784955007898467600689403773245L, 0.0L};
static const real WGK[8] = {
    0.022935322010529224963732008058970L, 0.063092092629978553290700663189204L,
    0.104790010322250183839876322541518L, 0.140653259715525918745189590510238L,
    0.169004726639267902826583426598550L, 0.190350578064785409913256402421014L,
    0.204432940075298892414161999234649L, 0.209482141084727828012999174891714L};
static const real WG[4] = {
    0.129484966168869693270611432679082L, 0.279705391489276667901467771423780L,
    0.381830050505118944950369775488975L, 0.417959183673469387755102040816327L};

template <class F>
static treal gk15(const F& f, treal a, treal b, treal& err) {
    const treal c = (a + b) / 2, h = (b - a) / 2;
    const treal fc = f(c);
    treal rk = WGK[7] * fc, rg = WG[3] * fc;
    for (int j = 0; j < 7; ++j) {
        const treal dx = h * XGK[j];
        const treal s = f(c - dx) + f(c + dx);
        rk += WGK[j] * s;
        if (j % 2 == 1) rg += WG[j / 2] * s;
    }
    err = std::fabs((rk - rg) * h);
    return rk * h;
}

template <class F>
static treal gk_refine(const F& f, treal a, treal b, treal whole, treal err, treal abs_tol, treal rel_tol,
                      int depth) {
    if (err <= abs_tol || err <= rel_tol * std::fabs(whole) || depth >= 48) return whole;
    const treal c = (a + b) / 2;
    treal e1, e2;
    const treal l = gk15(f, a, c, e1);
    const treal r = gk15(f, c, b, e2);
    return gk_refine(f, a, c, l, e1, abs_tol, rel_tol, depth + 1) +
           gk_refine(f, c, b, r, e2, abs_tol, rel_tol, depth + 1);
}

// integral of f over [a,b] to relative accuracy ~rel of the result
template <class F>
static treal integrate(const F& f, treal a, treal b, treal rel) {
    if (!(b > a)) return 0;
    treal e0;
    const treal i0 = gk15(f, a, b, e0);
    treal scale = std::fabs(i0);
    for (int pass = 0;; ++pass) {
        const treal v = gk_refine(f, a, b, i0, e0, rel * scale * 0.01, rel, 0);
        if (pass == 1 || std::fabs(v) >= 0.5 * scale) return v;
        scale = std::fabs(v);  // first estimate was far too large: tighten and redo
    }
}

// integral over consecutive panels given by sorted break points
template <class F>
static treal integrate_panels(const F& f, const std::vector<treal>& brk, treal rel) {
    treal s = 0;
    for (size_t i = 0; i + 1 < brk.size(); ++i) s += integrate(f, brk[i], brk[i + 1], rel);
    return s;
}

// -------------------------------------------------------------------------------------
//  Modified Bessel function of the second kind and its tail integral, exponentially
//  scaled:   Ks(nu,x)  = e^x K_nu(x)          = int_0^inf e^{-x(cosh t-1)} cosh(nu t) dt
//            IKs(nu,x) = e^x int_x^inf K_nu   = int_0^inf e^{-x(cosh t-1)} cosh(nu t)/cosh t dt
//  (DLMF 10.32.9, and the same with the s-integral of e^{-s cosh t} done in closed form).
// -------------------------------------------------------------------------------------
static const treal INNER_REL = 1e-13;  // on the Gauss-Kronrod error *estimate*; the true error is far smaller

// int_0^inf e^{-x(cosh t-1)} [ a cosh(nu_a t)/cosh t + b cosh(nu_b t) ] dt  =  a IKs(nu_a,x) + b Ks(nu_b,x)
static treal bessel_cosh_integral(treal x, treal a, treal nu_a, treal b, treal nu_b) {
    // cut where the integrand has dropped below e^{-45} of its value at t=0:
    // x(cosh t - 1) - nu t >= 45, solved with one fixed-point step
    const treal nu = std::max(a != 0 ? std::fabs(nu_a) : 0, b != 0 ? std::fabs(nu_b) : 0);
    const treal t0 = std::acosh(1 + 45 / x);
    const treal t_max = std::acosh(1 + (45 + nu * (t0 + 1)) / x);
    auto f = [&](treal t) {
        const treal sh = std::sinh(t / 2);  // cosh t - 1 = 2 sinh^2(t/2)
        treal w = 0;
        if (a != 0) w += a * std::cosh(nu_a * t) / std::cosh(t);
        if (b != 0) w += b * std::cosh(nu_b * t);
        return std::exp(-2 * x * sh * sh) * w;
    };
    const int npan = 3;
    treal s = 0;
    for (int i = 0; i < npan; ++i)
        s += integrate(f, t_max * i / npan, t_max * (i + 1) / npan, INNER_REL);
    return s;
}
static treal Ks(treal nu, treal x) { return bessel_cosh_integral(x, 0, 0, 1, nu); }
static treal IKs(treal nu, treal x) { return bessel_cosh_integral(x, 1, nu, 0, 0); }

// -------------------------------------------------------------------------------------
//  (I-a) Breit-Wheeler.  With xi = chi_-/chi_gamma, eq.5 gives chi_gamma X^{3/2} =
//  1/(xi(1-xi)) and (2/3)X^{3/2} = z := 2/(3 chi_gamma xi (1-xi)); substituting
//  t=(2/3)s^{3/2} turns int_X^inf sqrt(s) K_{1/3}((2/3)s^{3/2}) ds into int_z^inf K_{1/3}(t)dt.
//  Hence the bracket of eq.9 (the bracket of eq.4 at :90 is garbled) is
//      f_BW(chi_gamma, xi) = IK_{1/3}(z) - (2 - 1/(xi(1-xi))) K_{2/3}(z)
//  and  T = 1/(pi sqrt3 chi_gamma^2) int_0^chi_gamma [..] du = 1/(pi sqrt3 chi_gamma) int_0^1 f_BW dxi.
//  Everything is carried with e^{z0}, z0 = 8/(3 chi_gamma) = min_xi z, factored out, so that
//  chi_gamma down to 1e-4 (ln T ~ -26668) does not underflow (paper silent; R9).
// -------------------------------------------------------------------------------------
static treal bw_f_scaled(treal chi, treal xi) {  // e^{z0} f_BW
    if (!(xi > 0) || !(xi < 1)) return 0;
    const treal q = 1 / (xi * (1 - xi));
    const treal z = 2 * q / (3 * chi);
    const treal dz = 2 * (1 - 2 * xi) * (1 - 2 * xi) * q / (3 * chi);  // z - z0, no cancellation
    const treal e = std::exp(-dz);
    if (e == 0) return 0;
    return e * bessel_cosh_integral(z, 1, 1.0 / 3, -(2 - q), 2.0 / 3);  // IKs(1/3,z) - (2-q) Ks(2/3,z)
}

static std::vector<treal> bw_breaks(treal chi, treal lo, treal hi) {
    // the integrand is a bump of width sigma = sqrt(3 chi/64) around xi = 1/2 when chi << 1
    std::vector<treal> b = {lo, hi};
    const treal sigma = std::sqrt(3 * chi / 64);
    for (treal k = 1; k * sigma < 0.5; k *= 2) {
        for (treal s : {-1.0, 1.0}) {
            const treal x = 0.5 + s * k * sigma;
            if (x > lo && x < hi) b.push_back(x);
        }
    }
    if (0.5 > lo && 0.5 < hi) b.push_back(0.5);
    std::sort(b.begin(), b.end());
    return b;
}

static const treal OUTER_REL = 1e-11;  // on the error estimate, as above

static treal bw_integral_scaled(treal chi, treal lo, treal hi) {
    auto f = [&](treal xi) { return bw_f_scaled(chi, xi); };
    return integrate_panels(f, bw_breaks(chi, lo, hi), OUTER_REL);
}

// ln T(chi_gamma), eq.9
static treal bw_lnT(treal chi) {
    const treal I = bw_integral_scaled(chi, 0, 1);
    return std::log(I / (PI_L * std::sqrt(3.0) * chi)) - 8 / (3 * chi);
}

// -------------------------------------------------------------------------------------
//  (I-b) Photon emission (paper: "inverse Compton" / quantum synchrotron, QS).
//  eqs.12-14:  S(chi,xi)/xi = sqrt3/(2 pi) [ IK_{5/3}(Y) + xi^2/(1-xi) K_{2/3}(Y) ],
//  Y = 2 xi / (3 chi (1-xi)).  G(chi) = int_0^1 S/xi dxi (eq.16; the stray xi in the last
//  form of eq.17 is a typo, R3).
// -------------------------------------------------------------------------------------
static treal qs_s_over_xi(treal chi, treal xi) {
    if (!(xi > 0) || !(xi < 1)) return 0;
    const treal Y = 2 * xi / (3 * chi * (1 - xi));
    const treal e = std::exp(-Y);
    if (e == 0) return 0;
    return std::sqrt(3.0) / (2 * PI_L) * e *
           bessel_cosh_integral(Y, 1, 5.0 / 3, xi * xi / (1 - xi), 2.0 / 3);  // IKs(5/3,Y) + xi^2/(1-xi) Ks(2/3,Y)
}

// int_lo^hi S/xi dxi, by the substitution xi = v^3 (S/xi ~ xi^{-2/3} at xi -> 0 is then smooth)
static treal qs_integral_cuberoot(treal chi, treal lo, treal hi) {
    auto f = [&](treal v) { return 3 * v * v * qs_s_over_xi(chi, v * v * v); };
    std::vector<treal> b = {std::cbrt(lo), std::cbrt(hi)};
    for (treal Y : {1e-3, 1e-1, 1.0, 4.0, 16.0, 64.0, 256.0}) {
        const treal xi = 3 * chi * Y / (2 + 3 * chi * Y);  // where Y(chi,xi) = Y
        const treal v = std::cbrt(xi);
        if (v > b.front() && v < b[1]) b.push_back(v);
    }
    std::sort(b.begin(), b.end());
    return integrate_panels(f, b, OUTER_REL);
}
// the same integral taken literally in xi (used for the table cells, lo > 0)
static treal qs_integral_literal(treal chi, treal lo, treal hi) {
    auto f = [&](treal xi) { return qs_s_over_xi(chi, xi); };
    return integrate(f, lo, hi, OUTER_REL);
}

static treal qs_G(treal chi) { return qs_integral_cuberoot(chi, 0, 1); }

// -------------------------------------------------------------------------------------
//  Grids ("N points logarithmically distributed between
//  the extrema"; both ends included, R8).
// -------------------------------------------------------------------------------------
static treal log_grid(treal vmin, treal vmax, int n, int i) {
    if (i == 0) return vmin;
    if (i == n - 1) return vmax;
    return std::exp(std::log(vmin) + (std::log(vmax) - std::log(vmin)) * i / (n - 1));
}

// =====================================================================================
//  Exported: definitions (for pins) and table builders
// =====================================================================================
extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// max over k<=22 of | sum_j w_j x_j^k - int_{-1}^{1} x^k dx |  (Kronrod) and k<=13 (Gauss)
double orc_selftest_gk15() {
    treal worst = 0;
    for (int k = 0; k <= 22; ++k) {
        treal sk = 0, sg = 0;
        for (int j = 0; j < 8; ++j) {
            const treal p = std::pow(XGK[j], k);
            const treal both = (j == 7) ? p : p + (k % 2 ? -p : p);
            sk += WGK[j] * both;
            if (j % 2 == 1) sg += WG[j / 2] * both;
        }
        const treal exact = (k % 2) ? 0 : 2.0 / (k + 1);
        worst = std::max(worst, std::fabs(sk - exact));
        if (k <= 13) worst = std::max(worst, std::fabs(sg - exact));
    }
    return (double)worst;
}

double orc_schwinger_field() {  // eq.1, V/m
    return (double)(M_ELECTRON * M_ELECTRON * C_LIGHT * C_LIGHT * C_LIGHT / (Q_ELEM * hbar()));
}
double orc_rate_prefactor() { return (double)rate_prefactor(); }  // alpha m c^2 / hbar, 1/s

double orc_bessel_k_scaled(double nu, double x) { return (double)Ks(nu, x); }
double orc_bessel_ik_scaled(double nu, double x) { return (double)IKs(nu, x); }

double orc_bw_f_scaled(double chi, double xi) { return (double)bw_f_scaled(chi, xi); }
double orc_bw_lnT(double chi) { return (double)bw_lnT(chi); }
// e^{8/(3 chi)} T(chi)
double orc_bw_T_scaled(double chi) {
    return (double)(bw_integral_scaled(chi, 0, 1) / (PI_L * std::sqrt(3.0) * chi));
}
double orc_bw_cdf(double chi, double xi) {  // eq.11 in xi = chi_-/chi_gamma
    return (double)(bw_integral_scaled(chi, 0, xi) / bw_integral_scaled(chi, 0, 1));
}
double orc_qs_s_over_xi(double chi, double xi) { return (double)qs_s_over_xi(chi, xi); }
double orc_qs_G(double chi) { return (double)qs_G(chi); }
double orc_qs_cdf(double chi, double xi) {  // eq.18 as the number CDF (R4)
    return (double)(qs_integral_cuberoot(chi, 0, xi) / qs_G(chi));
}
// first moment int_0^1 S dxi (radiated power integrand; pin: -> chi^2 as chi -> 0)
double orc_qs_first_moment(double chi) {
    auto f = [&](treal v) { const treal xi = v * v * v; return 3 * v * v * xi * qs_s_over_xi(chi, xi); };
    return (double)integrate(f, 0, 1, OUTER_REL);
}

// ---- 1D tables: out[i] = ln T(chi_i) / ln G(chi_i), chi_i log-spaced incl. both ends ----
void orc_build_lnT(double chi_min, double chi_max, int n, double* out) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < n; ++i) out[i] = (double)bw_lnT(log_grid(chi_min, chi_max, n, i));
}
void orc_build_lnG(double chi_min, double chi_max, int n, double* out) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < n; ++i) out[i] = (double)std::log(qs_G(log_grid(chi_min, chi_max, n, i)));
}

// ---- 2D BW table: rows row0..row1-1 of P[n][m], xi_m = 0.5 m/(n_xi-1).
// Each row is a running sum of per-cell integrals (monotone by construction, R10)
// divided by the full integral over [0,1].  out has (row1-row0)*n_xi entries.
// half_check[r] (may be NULL) receives the computed P(chi,1/2) before it is fixed to 0.5.
void orc_build_bw_cdf_rows(double chi_min, double chi_max, int n_chi, int n_xi, int row0, int row1,
                           double* out, double* half_check) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int n = row0; n < row1; ++n) {
        const treal chi = log_grid(chi_min, chi_max, n_chi, n);
        std::vector<treal> cum(n_xi);
        cum[0] = 0;
        for (int m = 1; m < n_xi; ++m) {
            const treal lo = 0.5 * (m - 1) / (n_xi - 1), hi = 0.5 * m / (n_xi - 1);
            cum[m] = cum[m - 1] + bw_integral_scaled(chi, lo, hi);
        }
        const treal total = cum[n_xi - 1] + bw_integral_scaled(chi, 0.5, 1);
        double* row = out + (size_t)(n - row0) * n_xi;
        for (int m = 0; m < n_xi; ++m) row[m] = (double)(cum[m] / total);
        if (half_check) half_check[n - row0] = row[n_xi - 1];
        row[0] = 0.0;
        row[n_xi - 1] = 0.5;  // symmetry P(xi) = 1 - P(1-xi)
    }
}

// ---- 2D QS table: rows of ln P[n][m], xi_m = xi_min^{1 - m/(n_xi-1)}.
// g_check[r] (may be NULL) receives the row total (must equal G(chi_n)).
void orc_build_qs_cdf_rows(double chi_min, double chi_max, int n_chi, double xi_min, int n_xi,
                           int row0, int row1, double* out, double* g_check) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int n = row0; n < row1; ++n) {
        const treal chi = log_grid(chi_min, chi_max, n_chi, n);
        std::vector<treal> cum(n_xi);
        treal lo = xi_min;
        cum[0] = qs_integral_cuberoot(chi, 0, xi_min);
        for (int m = 1; m < n_xi; ++m) {
            const treal hi = log_grid(xi_min, 1.0, n_xi, m);
            cum[m] = cum[m - 1] + qs_integral_literal(chi, lo, hi);
            lo = hi;
        }
        const treal total = cum[n_xi - 1];
        double* row = out + (size_t)(n - row0) * n_xi;
        for (int m = 0; m < n_xi; ++m) row[m] = (double)std::log(cum[m] / total);
        if (g_check) g_check[n - row0] = (double)total;
    }
}

}  // extern "C"

// =====================================================================================
//  (II) Runtime half
// =====================================================================================

// ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  Pinned by the published
// known-answer vectors in tests/golden/philox4x32_10_kat.txt.
static inline void philox_round(uint32_t c[4], const uint32_t k[2]) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k[0];
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k[1];
    const uint32_t n3 = (uint32_t)p0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
}
static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]};
    uint32_t k[2] = {key[0], key[1]};
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }
        philox_round(c, k);
    }
    for (int i = 0; i < 4; ++i) out[i] = c[i];
}

// Stream layout (north star: "keyed on (seed, particle id, step)"):
// key = (seed_lo, seed_hi); counter = (id_lo, id_hi, step_lo, purpose | species<<8 | step_hi<<16).
// purpose 0: initial tau (words 0,1).  purpose 1: event (words 0,1 -> r; words 2,3 -> parent's new tau).
// purpose 2: children (words 0,1 -> tau of photon / electron; words 2,3 -> tau of positron).
static void qed_words(uint64_t seed, uint64_t id, uint64_t step, int purpose, int species,
                      uint32_t w[4]) {
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    const uint32_t ctr[4] = {(uint32_t)id, (uint32_t)(id >> 32), (uint32_t)step,
                             (uint32_t)purpose | ((uint32_t)species << 8) |
                                 ((uint32_t)((step >> 32) & 0xFFFFu) << 16)};
    philox4x32_10(ctr, key, w);
}
// uniform strictly inside (0,1), exact in the target type: fp64: (k+1/2) 2^-52, k = top 52 bits
// of (a:b); fp32: (k+1/2) 2^-23, k = a >> 9.
static real uniform_open(uint32_t a, uint32_t b, int dtype) {
    if (dtype == 1) {
        const uint64_t k = (((uint64_t)a << 32) | b) >> 12;
        return ((real)k + 0.5L) * 0x1p-52L;
    }
    const uint32_t k = a >> 9;
    return ((real)k + 0.5L) * 0x1p-23L;
}
static double round_to(real v, int dtype) { return dtype == 1 ? (double)v : (double)(float)v; }
// tau = -ln U  (tau "is extracted from p(x) = exp(-x)")
static double draw_tau(uint32_t a, uint32_t b, int tau_dtype) {
    return round_to(-logl(uniform_open(a, b, tau_dtype)), tau_dtype);
}

// ---- tables as the runtime sees them ----
struct OrcTables {
    double qs_chi_min, qs_chi_max; int qs_n_chi; double qs_xi_min; int qs_n_xi;
    double bw_chi_min, bw_chi_max; int bw_n_chi; int bw_n_xi;
    const double* lnG; const double* qs_lnP; const double* lnT; const double* bw_P;
    int read_fp32;  // 1: every table value is read through fp32 rounding
    // rows of the 2D tables when they sit on a chi grid of their own (0: the grid of the 1D table).  PAPER.md:203/:246 (1D)
    // and :210/:251 (2D) define the two grids separately; BASELINE configuration 4 asks for 4096 and 2048 points.
    int qs_n_chi_2d, bw_n_chi_2d;
    // PAPER.md:340 (WarpX): "a minimum quantum parameter threshold below which Breit-Wheeler pair production is ignored and
    // photon emission is simulated with a classical model" -- below chi_event_min neither process is an event (rate := 0;
    // DESIGN.md R24).  0 = off.  The classical model itself is orc_classical_loss below.
    double chi_event_min;
};
static inline int qs_rows(const OrcTables* t) { return t->qs_n_chi_2d > 0 ? t->qs_n_chi_2d : t->qs_n_chi; }
static inline int bw_rows(const OrcTables* t) { return t->bw_n_chi_2d > 0 ? t->bw_n_chi_2d : t->bw_n_chi; }
static inline real tab(const OrcTables* t, const double* a, size_t i) {
    return t->read_fp32 ? (real)(float)a[i] : (real)a[i];
}

// ---- chi, eqs.2-3 taken literally, in binary128, rounded once ----
// p in m_e c, e = E/E_s, b = cB/E_s.  With g = gamma (lepton) or |p| (photon):
// chi = sqrt( |g e + p x b|^2 - (p.e)^2 ).
static __float128 chi_q(int species, const double p[3], const double e[3], const double b[3],
                        __float128* g_out) {
    const __float128 px = p[0], py = p[1], pz = p[2];
    const __float128 p2 = px * px + py * py + pz * pz;
    const __float128 g = species == 0 ? sqrtq((__float128)1 + p2) : sqrtq(p2);
    const __float128 vx = g * e[0] + (py * b[2] - pz * b[1]);
    const __float128 vy = g * e[1] + (pz * b[0] - px * b[2]);
    const __float128 vz = g * e[2] + (px * b[1] - py * b[0]);
    const __float128 d = px * e[0] + py * e[1] + pz * e[2];
    __float128 c2 = vx * vx + vy * vy + vz * vz - d * d;
    if (c2 < 0) c2 = 0;
    if (g_out) *g_out = g;
    return sqrtq(c2);
}

// ---- 1D log-log lookup: eq.23 / eq.27.  Returns the interpolated ln value. ----
static real lookup_ln(const OrcTables* t, const double* L, real vmin, real vmax, int n, real lnchi,
                      real* slope_out) {
    const real lmin = logl(vmin), lmax = logl(vmax);
    const real delta = (lmax - lmin) / (n - 1);
    int k = (int)floorl((lnchi - lmin) / delta);
    k = std::max(0, std::min(n - 2, k));
    const real slope = (tab(t, L, k + 1) - tab(t, L, k)) / delta;
    if (slope_out) *slope_out = slope;
    return tab(t, L, k) + (lnchi - (lmin + k * delta)) * slope;
}

// Erber form used outside the T table (PAPER.md:203 -> eq.10 at :115, with the argument
// corrected to 4/(3 chi_gamma), R2):  T ~ 0.16 K_{1/3}(4/(3 chi))^2 / chi.
static real erber_T(real chi) {
    if (!(chi > 0)) return 0;
    const real x = 4 / (3 * chi);
    const real k = Ks(1.0L / 3, x);
    return 0.16L * k * k * expl(-2 * x) / chi;
}

// dN/dt in 1/s (eq.15 for leptons, eq.8 for photons); also the ln of the tabulated factor
static real qed_rate(const OrcTables* t, int species, real chi, real g, real* L_out, real* slope_out) {
    real L = 0, slope = 0, rate = 0;
    if (chi < (real)t->chi_event_min) {
        // below the threshold of PAPER.md:340: no event of either kind
    } else if (species == 0) {
        real lc = logl(chi);  // chi = 0 -> -inf -> clamped to the first value
        lc = std::max(logl((real)t->qs_chi_min), std::min(logl((real)t->qs_chi_max), lc));
        L = lookup_ln(t, t->lnG, t->qs_chi_min, t->qs_chi_max, t->qs_n_chi, lc, &slope);
        rate = (2.0L / 3) * rate_prefactor() * expl(L) / g;
    } else if (g > 2 && chi > 0) {  // photons with gamma_gamma <= 2 cannot decay (R12)
        real T;
        if (chi < t->bw_chi_min || chi > t->bw_chi_max) {
            T = erber_T(chi);
            L = T > 0 ? logl(T) : 0;
            slope = 4 / (3 * chi);
        } else {
            L = lookup_ln(t, t->lnT, t->bw_chi_min, t->bw_chi_max, t->bw_n_chi, logl(chi), &slope);
            T = expl(L);
        }
        rate = rate_prefactor() * chi * T / g;
    }
    if (L_out) *L_out = L;
    if (slope_out) *slope_out = slope;
    return rate;
}

// row bracket and weight for the 2D tables (chi clamped into the table)
static void row_bracket(real chi, real vmin, real vmax, int n, int* k_out, real* w_out) {
    const real lmin = logl(vmin), lmax = logl(vmax);
    const real lc = std::max(lmin, std::min(lmax, logl(chi)));
    const real delta = (lmax - lmin) / (n - 1);
    int k = (int)floorl((lc - lmin) / delta);
    k = std::max(0, std::min(n - 2, k));
    *k_out = k;
    *w_out = (lc - (lmin + k * delta)) / delta;
}

// eqs.28-30: xi = chi_gamma/chi of the emitted photon for uniform r
static real qs_sample_xi(const OrcTables* t, real chi, real r) {
    int k; real w;
    row_bracket(chi, t->qs_chi_min, t->qs_chi_max, qs_rows(t), &k, &w);
    const int M = t->qs_n_xi;
    const double* r0 = t->qs_lnP + (size_t)k * M;
    const double* r1 = r0 + M;
    auto ell = [&](int m) { return tab(t, r0, m) + w * (tab(t, r1, m) - tab(t, r0, m)); };  // eq.28
    const real lr = logl(r);
    const real lxi_min = logl((real)t->qs_xi_min);
    if (lr < ell(0)) return t->qs_xi_min;  // below the first column (paper silent; R6)
    int lo = 0, hi = M - 1;                // invariant: ell(lo) <= lr; answer = max{m: ell(m) <= lr}
    while (hi - lo > 1) {                  // binary search, eq.29
        const int mid = (lo + hi) / 2;
        if (ell(mid) <= lr) lo = mid; else hi = mid;
    }
    if (ell(hi) <= lr) lo = hi;
    const int ms = std::min(lo, M - 2);
    auto lxi = [&](int m) { return lxi_min * (1 - (real)m / (M - 1)); };
    const real a = ell(ms), b = ell(ms + 1);
    if (!(b > a)) return expl(lxi(ms));
    return expl(lxi(ms) + (lr - a) * (lxi(ms + 1) - lxi(ms)) / (b - a));  // eq.30
}

// eqs.24-26 on r' = min(r, 1-r) in [0, 1/2]: xi = chi/chi_gamma in [0, 1/2]
static real bw_sample_xi(const OrcTables* t, real chi, real rp) {
    int k; real w;
    row_bracket(chi, t->bw_chi_min, t->bw_chi_max, bw_rows(t), &k, &w);
    const int M = t->bw_n_xi;
    const double* r0 = t->bw_P + (size_t)k * M;
    const double* r1 = r0 + M;
    auto P = [&](int m) { return tab(t, r0, m) + w * (tab(t, r1, m) - tab(t, r0, m)); };  // eq.24
    int lo = 0, hi = M - 1;  // P(0) = 0 <= r'
    while (hi - lo > 1) {    // binary search, eq.25
        const int mid = (lo + hi) / 2;
        if (P(mid) <= rp) lo = mid; else hi = mid;
    }
    if (P(hi) <= rp) lo = hi;
    const int ms = std::min(lo, M - 2);
    auto xi = [&](int m) { return 0.5L * m / (M - 1); };
    const real a = P(ms), b = P(ms + 1);
    if (!(b > a)) return xi(ms);
    return xi(ms) + (rp - a) * (xi(ms + 1) - xi(ms)) / (b - a);  // eq.26
}

extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    philox4x32_10(ctr, key, out);
}
// the uniform the method draws: pair = 0 -> words (0,1), pair = 1 -> words (2,3)
double orc_uniform(uint64_t seed, uint64_t id, uint64_t step, int purpose, int species, int pair,
                   int dtype) {
    uint32_t w[4];
    qed_words(seed, id, step, purpose, species, w);
    return (double)uniform_open(w[2 * pair], w[2 * pair + 1], dtype);
}

// chi for n particles (inputs as doubles; fp32 inputs are passed widened, which is exact)
void orc_chi(int species, int64_t n, const double* px, const double* py, const double* pz,
             const double* ex, const double* ey, const double* ez, const double* bx,
             const double* by, const double* bz, double* chi_out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double p[3] = {px[i], py[i], pz[i]}, e[3] = {ex[i], ey[i], ez[i]},
                     b[3] = {bx[i], by[i], bz[i]};
        chi_out[i] = (double)chi_q(species, p, e, b, nullptr);
    }
}

// tau = -ln U, purpose 0, step 0
void orc_init_optical_depth(int species, int tau_dtype, int64_t n, uint64_t seed,
                            const uint64_t* ids, double* tau) {
    for (int64_t i = 0; i < n; ++i) {
        uint32_t w[4];
        qed_words(seed, ids[i], 0, 0, species, w);
        tau[i] = draw_tau(w[0], w[1], tau_dtype);
    }
}

// rate only (1/s) -- used by the harness to choose dt, and by the Monte Carlo pins
void orc_rate(const OrcTables* t, int species, int64_t n, const double* px, const double* py,
              const double* pz, const double* ex, const double* ey, const double* ez,
              const double* bx, const double* by, const double* bz, double* rate_out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double p[3] = {px[i], py[i], pz[i]}, e[3] = {ex[i], ey[i], ez[i]},
                     b[3] = {bx[i], by[i], bz[i]};
        __float128 g;
        const real chi = (real)chi_q(species, p, e, b, &g);
        rate_out[i] = (double)qed_rate(t, species, chi, (real)g, nullptr, nullptr);
    }
}

// tau <- tau - dN/dt dt.  tau_out is rounded to tau_dtype; tau_exact (may be
// NULL) keeps the unrounded long-double value as a double, decr / lnval / slope (may be NULL)
// are the decrement, the interpolated ln T or ln G and d ln(value)/d ln(chi), from which the
// tests build the tie margin.
void orc_evolve_optical_depth(const OrcTables* t, int species, int tau_dtype, int64_t n,
                              const double* px, const double* py, const double* pz,
                              const double* ex, const double* ey, const double* ez,
                              const double* bx, const double* by, const double* bz, double dt,
                              const double* tau_in, double* tau_out, double* tau_exact,
                              double* decr, double* lnval, double* slope) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double p[3] = {px[i], py[i], pz[i]}, e[3] = {ex[i], ey[i], ez[i]},
                     b[3] = {bx[i], by[i], bz[i]};
        __float128 g;
        const real chi = (real)chi_q(species, p, e, b, &g);
        real L, sl;
        const real rate = qed_rate(t, species, chi, (real)g, &L, &sl);
        const real d = rate * (real)dt;
        const real tn = (real)tau_in[i] - d;
        tau_out[i] = round_to(tn, tau_dtype);
        if (tau_exact) tau_exact[i] = (double)tn;
        if (decr) decr[i] = (double)d;
        if (lnval) lnval[i] = (double)L;
        if (slope) slope[i] = (double)sl;
    }
}

// Classical radiation reaction below the threshold of PAPER.md:340 (R24; refs [58, 59] of the paper are not in
// the container).  Reading: a lepton with chi < chi_min loses energy continuously at the classical radiated power, which
// is the chi -> 0 limit of the mean loss of the Monte Carlo emission: the emission rate (2/3)(alpha/tau_C) G/gamma (eq.15)
// times the mean photon energy (gamma - 1) <xi>, <xi> = int S dxi / G, with int S dxi -> chi^2 (classical synchrotron power):
//     d(gamma - 1)/dt = -(2/3) (alpha/tau_C) chi^2 (gamma - 1)/gamma,
// one explicit step per call, direction kept, norm(p') from gamma' (as for an emission, R15), the kinetic energy
// not below zero.  Leptons at or above the threshold are left alone.
void orc_classical_loss(int dtype, int64_t n, double* px, double* py, double* pz, const double* ex, const double* ey,
                        const double* ez, const double* bx, const double* by, const double* bz, double dt,
                        double chi_min) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double p[3] = {px[i], py[i], pz[i]}, e[3] = {ex[i], ey[i], ez[i]}, b[3] = {bx[i], by[i], bz[i]};
        __float128 gq;
        const real chi = (real)chi_q(0, p, e, b, &gq);
        if (!(chi < (real)chi_min)) continue;
        const real g = (real)gq;
        const real pn = sqrtl((real)p[0] * p[0] + (real)p[1] * p[1] + (real)p[2] * p[2]);
        if (!(pn > 0)) continue;
        const real k = pn * pn / (g + 1);  // gamma - 1
        real k2 = k - (2.0L / 3) * rate_prefactor() * chi * chi * (k / g) * (real)dt;
        if (k2 < 0) k2 = 0;
        const real s = sqrtl(k2 * (k2 + 2)) / pn;
        px[i] = round_to(s * p[0], dtype);
        py[i] = round_to(s * p[1], dtype);
        pz[i] = round_to(s * p[2], dtype);
    }
}

// Photon emission for leptons with tau < 0.  Serial loop in index
// order: this loop *defines* the order of the secondaries.  The first `capacity` fired
// parents are processed; later ones are left untouched (tau stays negative).  Returns the
// number of fired parents (which may exceed capacity).  p and tau are updated in place.
int64_t orc_generate_photons(const OrcTables* t, int dtype, int tau_dtype, int64_t n, double* px,
                             double* py, double* pz, const double* ex, const double* ey,
                             const double* ez, const double* bx, const double* by,
                             const double* bz, double* tau, uint64_t seed, uint64_t step,
                             const uint64_t* ids, int64_t capacity, double* ph_px, double* ph_py,
                             double* ph_pz, double* ph_tau, int64_t* ph_parent, double* ph_xi) {
    int64_t n_out = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (!(tau[i] < 0)) continue;  // event <=> tau < 0 (R1)
        const int64_t slot = n_out++;
        if (slot >= capacity) continue;
        const double p[3] = {px[i], py[i], pz[i]}, e[3] = {ex[i], ey[i], ez[i]},
                     b[3] = {bx[i], by[i], bz[i]};
        __float128 gq;
        const real chi = (real)chi_q(0, p, e, b, &gq);
        const real g = (real)gq;
        uint32_t w[4], wc[4];
        qed_words(seed, ids[i], step, 1, 0, w);
        qed_words(seed, ids[i], step, 2, 0, wc);
        const real r = uniform_open(w[0], w[1], dtype);
        const real xi = qs_sample_xi(t, chi, r);
        const real gph = (g - 1) * xi;  // gamma_gamma = (gamma-1) xi
        const real pn = sqrtl((real)p[0] * p[0] + (real)p[1] * p[1] + (real)p[2] * p[2]);
        const real nx = p[0] / pn, ny = p[1] / pn, nz = p[2] / pn;
        const real g2 = g - gph;        // kinetic energy reduced by gamma_gamma m c^2
        const real pn2 = sqrtl((g2 - 1) * (g2 + 1));
        ph_px[slot] = round_to(gph * nx, dtype);  // emitted along p
        ph_py[slot] = round_to(gph * ny, dtype);
        ph_pz[slot] = round_to(gph * nz, dtype);
        ph_tau[slot] = draw_tau(wc[0], wc[1], tau_dtype);
        if (ph_parent) ph_parent[slot] = i;
        if (ph_xi) ph_xi[slot] = (double)xi;
        px[i] = round_to(pn2 * nx, dtype);
        py[i] = round_to(pn2 * ny, dtype);
        pz[i] = round_to(pn2 * nz, dtype);
        tau[i] = draw_tau(w[2], w[3], tau_dtype);
    }
    return n_out;
}

// Pair production for photons with tau < 0.  Same ordering and
// capacity rule.  The photon is marked dead: p = 0, tau = +inf.
int64_t orc_generate_pairs(const OrcTables* t, int dtype, int tau_dtype, int64_t n, double* px,
                           double* py, double* pz, const double* ex, const double* ey,
                           const double* ez, const double* bx, const double* by, const double* bz,
                           double* tau, uint64_t seed, uint64_t step, const uint64_t* ids,
                           int64_t capacity, double* el_px, double* el_py, double* el_pz,
                           double* el_tau, double* po_px, double* po_py, double* po_pz,
                           double* po_tau, int64_t* parent, double* xi_el) {
    int64_t n_out = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (!(tau[i] < 0)) continue;
        const int64_t slot = n_out++;
        if (slot >= capacity) continue;
        const double p[3] = {px[i], py[i], pz[i]}, e[3] = {ex[i], ey[i], ez[i]},
                     b[3] = {bx[i], by[i], bz[i]};
        __float128 gq;
        const real chi = (real)chi_q(1, p, e, b, &gq);
        const real g = (real)gq;  // gamma_gamma = |p|
        uint32_t w[4], wc[4];
        qed_words(seed, ids[i], step, 1, 1, w);
        qed_words(seed, ids[i], step, 2, 1, wc);
        const real r = uniform_open(w[0], w[1], dtype);
        const bool electron_side = (r <= 0.5L);  // PAPER.md:212 "If r <= 0.5"
        const real rp = electron_side ? r : 1 - r;
        const real xi = bw_sample_xi(t, chi, rp);
        const real xe = electron_side ? xi : 1 - xi;  // chi_-/chi_gamma
        const real xp = electron_side ? 1 - xi : xi;  // chi_+/chi_gamma, eq.6
        const real ge = 1 + (g - 2) * xe;  // K = (gamma_gamma - 2) chi_pm/chi_gamma
        const real gp = 1 + (g - 2) * xp;
        const real nx = p[0] / g, ny = p[1] / g, nz = p[2] / g;
        const real pe = sqrtl((ge - 1) * (ge + 1)), pp = sqrtl((gp - 1) * (gp + 1));
        el_px[slot] = round_to(pe * nx, dtype);
        el_py[slot] = round_to(pe * ny, dtype);
        el_pz[slot] = round_to(pe * nz, dtype);
        po_px[slot] = round_to(pp * nx, dtype);
        po_py[slot] = round_to(pp * ny, dtype);
        po_pz[slot] = round_to(pp * nz, dtype);
        el_tau[slot] = draw_tau(wc[0], wc[1], tau_dtype);
        po_tau[slot] = draw_tau(wc[2], wc[3], tau_dtype);
        if (parent) parent[slot] = i;
        if (xi_el) xi_el[slot] = (double)xe;
        px[i] = 0; py[i] = 0; pz[i] = 0;
        tau[i] = std::numeric_limits<double>::infinity();
    }
    return n_out;
}

// ---- Schwinger pair production rate per unit volume (eqs.19-22), SURVEY.md 8(f)-3 ----
// Fields in units of E_s (e = E/E_s, b = cB/E_s).  Invariants F = (e^2 - b^2)/2, G = e.b (eqs.21-22, in E_s^2),
// epsilon = sqrt(sqrt(F^2+G^2) + F), eta = sqrt(sqrt(F^2+G^2) - F) (eq.20), and eq.19 taken literally in
// binary128 (the difference under the second root cancels when F >> abs(G)):
//     d^2N/dt dV = q_e^2 E_s^2/(4 pi^2 hbar^2 c) * epsilon eta coth(pi eta/epsilon) exp(-pi/epsilon)   [1/(m^3 s)]
// eta -> 0 is the removable limit eta coth(pi eta/epsilon) -> epsilon/pi; epsilon = 0 gives 0.
static real schwinger_prefactor() {
    const real es = M_ELECTRON * M_ELECTRON * C_LIGHT * C_LIGHT * C_LIGHT / (Q_ELEM * hbar());
    return Q_ELEM * Q_ELEM * es * es / (4 * PI_L * PI_L * hbar() * hbar() * C_LIGHT);
}
double orc_schwinger_prefactor() { return (double)schwinger_prefactor(); }
void orc_schwinger_rate(int64_t n, const double* ex, const double* ey, const double* ez, const double* bx,
                        const double* by, const double* bz, double* rate_out) {
    const __float128 PIq = 4 * atanq((__float128)1);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const __float128 e2 = (__float128)ex[i] * ex[i] + (__float128)ey[i] * ey[i] + (__float128)ez[i] * ez[i];
        const __float128 b2 = (__float128)bx[i] * bx[i] + (__float128)by[i] * by[i] + (__float128)bz[i] * bz[i];
        const __float128 F = (e2 - b2) / 2;
        const __float128 G = (__float128)ex[i] * bx[i] + (__float128)ey[i] * by[i] + (__float128)ez[i] * bz[i];
        const __float128 root = sqrtq(F * F + G * G);
        __float128 eps2 = root + F, eta2 = root - F;
        if (eps2 < 0) eps2 = 0;
        if (eta2 < 0) eta2 = 0;
        const __float128 eps = sqrtq(eps2), eta = sqrtq(eta2);
        __float128 r = 0;
        if (eps > 0) {
            const __float128 x = PIq * eta / eps;
            const __float128 eta_coth = x > (__float128)1e-12 ? eta * (coshq(x) / sinhq(x)) : eps / PIq;  // removable limit
            r = eps * eta_coth * expq(-PIq / eps);
        }
        rate_out[i] = (double)((__float128)schwinger_prefactor() * r);
    }
}

// the inverse-CDF maps alone (for the distribution pins)
double orc_qs_sample_xi(const OrcTables* t, double chi, double r) {
    return (double)qs_sample_xi(t, chi, r);
}
double orc_bw_sample_xi(const OrcTables* t, double chi, double rp) {
    return (double)bw_sample_xi(t, chi, rp);
}
double orc_erber_T(double chi) { return (double)erber_T(chi); }

}  // extern "C"
