// =====================================================================================
//  qed_device.cuh -- device-side building blocks of the PICSAR-QED hot path (sm_100a).
//
//  chi (PAPER.md:70 eq.2, :77 eq.3), 1D log-log table lookups (eq.23,
//  :248 eq.27), the Erber form outside the T table (PAPER.md:115 eq.10, :203), the
//  inverse-CDF lookups (PAPER.md:214-230 eqs.24-26, :257-267 eqs.28-30), Philox4x32-10
//  uniforms.  Product code: shares nothing with oracle/.
// =====================================================================================
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pxq {

// ---- physical constants (CODATA 2018; R14) --------------------------------
// alpha m_e c^2 / hbar in 1/s: prefactor of eq.8 and eq.15.
constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kFineStructure = 7.2973525693e-3;
constexpr double kElectronMass = 9.1093837015e-31;  // kg
constexpr double kLightSpeed = 299792458.0;         // m/s
constexpr double kPlanck = 6.62607015e-34;          // J s
constexpr double kAlphaOverTauC =
    kFineStructure * kElectronMass * kLightSpeed * kLightSpeed / (kPlanck / (2.0 * kPi));  // 5.6652563985e18

// ---- unit system of the caller's arrays ---------------------------------
// Multipliers that take the caller's momenta, electric and magnetic fields to the library's units (p/(m_e c), E/E_s,
// cB/E_s), applied in registers where the arrays are loaded; inv_p takes momenta back where they are stored.
// All 1 for the library's own units: x * 1.0 is exact, results are bit-identical to unscaled code.
struct UnitScales {
    double p = 1.0, e = 1.0, b = 1.0, inv_p = 1.0;
};

// ---- table views: plain structs passed by value to the kernels ----
template <typename R>
struct Table1D {      // ln G or ln T on a log-spaced chi grid
    const R* L;       // n values
    int n;
    double ln_min;    // ln chi_0
    double ln_max;    // ln chi_{n-1}
    double inv_delta; // (n-1)/(ln_max - ln_min)
    double chi_min, chi_max;
    double c2_event_min;  // square of the chi threshold of PAPER.md:340 (picsarqed_set_chi_threshold; 0 = off): no event below
};

template <typename R>
struct Table2D {      // rows: log-spaced chi; columns: xi grid
    const R* P;       // n_chi * n_xi, row-major
    int n_chi, n_xi;
    double ln_min, ln_max, inv_delta;
    double ln_xi_min; // QS only: ln(xi_min)
    double xi_step;   // column spacing: ln xi_{m+1} - ln xi_m (QS), xi_{m+1} - xi_m (BW); the host's division
    // search guide (may be null): guide[n * (bins + 1) + j] = max{m : P[n][m] <= key_j} (0 if none, and for j = 0),
    // key_j = guide_k0 + j / guide_inv_dk: narrows the binary search of eq.25 / eq.29 without changing its result
    const unsigned short* guide;
    int guide_bins;
    int guide_split;  // 1 (photon emission): lower half of the bins uniform in ln r on [guide_k0, ln 1/2], upper half uniform in r on [1/2, 1]
    double guide_k0, guide_inv_dk;
};

// ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) --------------------------------
struct Words4 { uint32_t w[4]; };

__device__ __forceinline__ Words4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                uint32_t k0, uint32_t k1) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += W0;
        k1 += W1;
    }
    Words4 o;
    o.w[0] = c0; o.w[1] = c1; o.w[2] = c2; o.w[3] = c3;
    return o;
}

// counter layout: (id_lo, id_hi, step_lo, purpose | species<<8 | step_hi16<<16)
__device__ __forceinline__ Words4 qed_words(uint64_t seed, uint64_t id, uint64_t step, int purpose, int species) {
    const uint32_t c3 = (uint32_t)purpose | ((uint32_t)species << 8) | ((uint32_t)((step >> 32) & 0xFFFFu) << 16);
    return philox4x32_10((uint32_t)id, (uint32_t)(id >> 32), (uint32_t)step, c3, (uint32_t)seed,
                         (uint32_t)(seed >> 32));
}

// uniform strictly inside (0,1), exact in the target type.
template <typename T> __device__ __forceinline__ T uniform_open(uint32_t a, uint32_t b);
template <> __device__ __forceinline__ double uniform_open<double>(uint32_t a, uint32_t b) {
    const uint64_t k = (((uint64_t)a << 32) | b) >> 12;          // top 52 bits
    return ((double)(long long)k + 0.5) * 0x1p-52;               // k < 2^52: exact
}
template <> __device__ __forceinline__ float uniform_open<float>(uint32_t a, uint32_t) {
    return ((float)(a >> 9) + 0.5f) * 0x1p-23f;                  // k < 2^23: exact
}
// ---- lean fp64 elementary functions for the streaming kernel ------------------------------------
// The CUDA library log/exp cost ~85 / ~50 instructions per call (special cases, constant moves); in the evolve
// kernel they were 45 % of all instructions (round-1 capture).  These versions assume what holds
// there -- log of a positive normal number (anything else takes the library path), exp of a finite argument --
// and keep the error at the 1e-16 level: a few ulp, far inside the 1e-9 tolerance on the optical depth.
// They are written for V arguments at once (log_pos_v, exp_fast_v; the scalar names are V = 1): the common path is one
// straight line for all V, so that the compiler interleaves the V dependent chains, and the special cases are selects
// or one rarely taken branch at the end.  The polynomial coefficients live in constant memory: an FMA takes them as a
// constant-bank operand, where an immediate costs two moves per use.
__constant__ double kLogCoef[9] = {1.0 / 19.0, 1.0 / 17.0, 1.0 / 15.0, 1.0 / 13.0, 1.0 / 11.0, 1.0 / 9.0, 1.0 / 7.0, 1.0 / 5.0, 1.0 / 3.0};
__constant__ double kExpCoef[12] = {1.0 / 6227020800.0, 1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0,
                                    1.0 / 40320.0, 1.0 / 5040.0, 1.0 / 720.0, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0, 0.5};
__constant__ double kLn2[3] = {6.93147180369123816490e-01, 1.90821492927058770002e-10, 1.4426950408889634074};  // hi, lo, log2(e)

__device__ __forceinline__ double rcp_fast(double x) {        // 1/x for normal x, ~1 ulp
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));     // ~20 bits
    r = fma(fma(-x, r, 1.0), r, r);                           // ~40 bits
    return fma(fma(-x, r, 1.0), r, r);                        // ~80 bits -> rounded
}
__device__ __forceinline__ double rsqrt_fast(double x) {      // 1/sqrt(x) for normal x > 0, ~1 ulp
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));   // ~20 bits
    const double hx = 0.5 * x;
    y = fma(fma(-hx * y, y, 0.5), y, y);
    return fma(fma(-hx * y, y, 0.5), y, y);
}
// ln x for positive normal x; anything else (zero, denormal, inf, nan, negative) takes the library routine
template <int V>
__device__ __forceinline__ void log_pos_v(const double (&x)[V], double (&y)[V]) {
    double s[V], s2[V], p[V], ed[V];
    bool special = false;
#pragma unroll
    for (int v = 0; v < V; ++v) {
        int hi = __double2hiint(x[v]);
        const int lo = __double2loint(x[v]);
        special = special || (unsigned)(hi - 0x00100000) >= 0x7fe00000u;
        int e = (hi >> 20) - 1023;
        hi = (hi & 0x000fffff) | 0x3ff00000;                 // mantissa in [1, 2)
        const bool up = hi >= 0x3ff6a09e;                    // -> [sqrt(1/2), sqrt(2))
        hi = up ? hi - 0x00100000 : hi;
        e = up ? e + 1 : e;
        ed[v] = (double)e;
        const double m = __hiloint2double(hi, lo);
        const double num = m - 1.0, den = m + 1.0;
        const double r = rcp_fast(den);
        const double s0 = num * r;
        s[v] = fma(fma(-s0, den, num), r, s0);               // s = (m-1)/(m+1), |s| <= 0.1716
        s2[v] = s[v] * s[v];
        p[v] = kLogCoef[0];
    }
    // ln m = 2 atanh(s) = 2 s (1 + s^2/3 + s^4/5 + ... + s^18/19); the first dropped term is < 3e-17
#pragma unroll
    for (int k = 1; k < 9; ++k)
#pragma unroll
        for (int v = 0; v < V; ++v) p[v] = fma(p[v], s2[v], kLogCoef[k]);
#pragma unroll
    for (int v = 0; v < V; ++v) {
        const double two_s = s[v] + s[v];
        const double lnm = fma(two_s * s2[v], p[v], two_s);
        y[v] = fma(ed[v], kLn2[0], fma(ed[v], kLn2[1], lnm));   // e ln2 (hi + lo)
    }
    if (special) {
#pragma unroll
        for (int v = 0; v < V; ++v)
            if ((unsigned)(__double2hiint(x[v]) - 0x00100000) >= 0x7fe00000u) y[v] = log(x[v]);
    }
}
// e^x for any x (0 below -707, e^709 above 709, nan for nan)
template <int V>
__device__ __forceinline__ void exp_fast_v(const double (&x)[V], double (&y)[V]) {
    double r[V], p[V];
    int k[V];
#pragma unroll
    for (int v = 0; v < V; ++v) {
        double xc = x[v] > 709.0 ? 709.0 : x[v];
        xc = xc > -707.0 ? xc : -707.0;                      // (keeps k in range; the result is replaced below)
        const double t = fma(xc, kLn2[2], 6755399441055744.0);   // k = rint(x log2 e) in the low word
        k[v] = __double2loint(t);
        const double kd = t - 6755399441055744.0;
        r[v] = fma(kd, -kLn2[1], fma(kd, -kLn2[0], xc));     // |r| <= 0.3466
        p[v] = kExpCoef[0];                                  // Taylor to r^13/13!: remainder < 2e-17
    }
#pragma unroll
    for (int j = 1; j < 12; ++j)
#pragma unroll
        for (int v = 0; v < V; ++v) p[v] = fma(p[v], r[v], kExpCoef[j]);
#pragma unroll
    for (int v = 0; v < V; ++v) {
        p[v] = fma(p[v], r[v], 1.0);
        p[v] = fma(p[v], r[v], 1.0);
        const double e = __hiloint2double(__double2hiint(p[v]) + (k[v] << 20), __double2loint(p[v]));  // p 2^k, k in [-1021, 1023]
        y[v] = x[v] > -707.0 ? e : (x[v] < 0.0 ? 0.0 : x[v]);   // underflow (or nan)
    }
}
__device__ __forceinline__ double log_pos(double x) {
    const double a[1] = {x};
    double y[1];
    log_pos_v<1>(a, y);
    return y[0];
}
__device__ __forceinline__ double exp_fast(double x) {
    const double a[1] = {x};
    double y[1];
    exp_fast_v<1>(a, y);
    return y[0];
}

// tau = -ln U
template <typename T> __device__ __forceinline__ T draw_tau(uint32_t a, uint32_t b);
template <> __device__ __forceinline__ double draw_tau<double>(uint32_t a, uint32_t b) {
    return -log_pos(uniform_open<double>(a, b));   // (u is a positive normal number: the lean logarithm applies)
}
template <> __device__ __forceinline__ float draw_tau<float>(uint32_t a, uint32_t b) {
    return -logf(uniform_open<float>(a, b));
}

// ---- chi^2 --------------------------------------------------------------------------
// eq.2 / eq.3: chi^2 = |g e + p x b|^2 - (p.e)^2.  Taken literally the two terms cancel by
// up to gamma^2 when e has a component along p, so it is evaluated in the equivalent form
//     chi^2 = |g e_perp + p x b|^2 + (g^2 - p^2) (e.p)^2 / p^2,   e_perp = e - (e.p) p / p^2,
// (g^2 - p^2 = 1 for leptons, 0 for photons), always in fp64 registers.
// Returns chi^2; *g2_out = g^2 (= 1 + p^2 or p^2).
template <int SPECIES>
__device__ __forceinline__ double chi_squared(double px, double py, double pz, double ex, double ey, double ez,
                                              double bx, double by, double bz, double g, double q) {   // q = 1/p^2 (0 for p = 0)
    const double d = fma(px, ex, fma(py, ey, pz * ez));  // p.e
    const double t = d * q;
    const double fx = fma(-t, px, ex), fy = fma(-t, py, ey), fz = fma(-t, pz, ez);  // e_perp
    const double cx = fma(py, bz, -pz * by), cy = fma(pz, bx, -px * bz), cz = fma(px, by, -py * bx);
    const double vx = fma(g, fx, cx), vy = fma(g, fy, cy), vz = fma(g, fz, cz);
    double c2 = fma(vx, vx, fma(vy, vy, vz * vz));
    if (SPECIES == 0) c2 = fma(d, t, c2);  // + (e.n)^2
    return c2;
}

// chi^2 with g and 1/g from one fast reciprocal square root: the one routine both passes use, so that the
// evolve pass and the event pass see bit-identical chi for the same particle
template <int SPECIES>
__device__ __forceinline__ double chi_squared_of(double px, double py, double pz, double ex, double ey, double ez,
                                                 double bx, double by, double bz, double* inv_g_out, double* g2_out) {
    const double p2 = fma(px, px, fma(py, py, pz * pz));
    const double g2 = SPECIES == 0 ? 1.0 + p2 : p2;
    const double inv_g = g2 > 1e-300 ? rsqrt_fast(g2) : 0.0;  // 1/gamma (lepton) or 1/gamma_gamma (photon)
    *inv_g_out = inv_g;
    *g2_out = g2;
    // 1/p^2: a photon's is (1/gamma_gamma)^2, the reciprocal square root squared (one multiplication)
    const double q = SPECIES == 1 ? inv_g * inv_g : (p2 > 1e-300 ? rcp_fast(p2) : 0.0);
    return chi_squared<SPECIES>(px, py, pz, ex, ey, ez, bx, by, bz, g2 * inv_g, q);
}

// ---- K_{1/3}(x), only for the Erber branch outside the T table -------------------------
// returns ln K_{1/3}(x) + x  (exponentially scaled, so chi_gamma -> 0 does not underflow)
__device__ __noinline__ double ln_bessel_k13_scaled(double x) {
    const double nu = 1.0 / 3.0;
    if (x >= 25.0) {  // Hankel asymptotic expansion (DLMF 10.40.2); terms fall below 1e-17 before they grow
        const double mu = 4.0 * nu * nu;
        double term = 1.0, sum = 1.0;
        const double r = 1.0 / (8.0 * x);
        for (int k = 1; k <= 24; ++k) {
            const double o = 2.0 * k - 1.0;
            term *= (mu - o * o) * r / k;
            sum += term;
            if (fabs(term) < 1e-17) break;
        }
        return 0.5 * log(1.5707963267948966 / x) + log(sum);
    }
    if (x <= 2.0) {  // ascending series: K = (pi/2)(I_{-nu} - I_nu)/sin(nu pi) (DLMF 10.27.4, 10.25.2)
        const double y = 0.25 * x * x;
        double tm = 1.0 / 1.3541179394264004;  // 1/Gamma(2/3):  I_{-1/3} term k = 0
        double tp = 1.0 / 0.8929795115692492;  // 1/Gamma(4/3):  I_{+1/3} term k = 0
        double sm = tm, sp = tp;
        for (int k = 1; k <= 30; ++k) {
            tm *= y / (k * (k - nu));
            tp *= y / (k * (k + nu));
            sm += tm;
            sp += tp;
            if (tm < 1e-18 * sm) break;
        }
        const double h = cbrt(0.5 * x);
        const double kv = 1.5707963267948966 / 0.8660254037844386 * (sm / h - sp * h);
        return log(kv) + x;
    }
    // 2 < x < 25: trapezoid rule on e^x K_nu(x) = int_0^inf exp(-2x sinh^2(t/2)) cosh(nu t) dt (DLMF 10.32.9)
    const double h = fmin(0.1, 0.35 * rsqrt(x));
    double s = 0.5;
    for (int j = 1; j < 400; ++j) {
        const double t = j * h;
        const double sh = sinh(0.5 * t);
        const double a = 2.0 * x * sh * sh;
        if (a > 46.0) break;
        s += exp(-a) * cosh(nu * t);
    }
    return log(s * h);
}

// ln of the tabulated factor times chi^POW... see lookup_ln_rate below.
// 1D log-log lookup (eq.23 / eq.27): returns the interpolated ln value at ln chi = lc
// (lc must already be inside [ln_min, ln_max]).  `tab` may live in shared memory.
template <typename R, typename A>
__device__ __forceinline__ A lookup_ln(const R* tab, int n, A lc, A ln_min, A inv_delta) {
    const A t = (lc - ln_min) * inv_delta;
    int k = (int)t;  // t >= 0
    k = min(k, n - 2);
    const A f = t - (A)k;
    const A l0 = (A)tab[k], l1 = (A)tab[k + 1];
    return fma(f, l1 - l0, l0);
}

// row bracket of the 2D tables (chi clamped into the table)
template <typename R>
__device__ __forceinline__ void row_bracket(const Table2D<R>& T, double ln_chi, int* k_out, double* w_out) {
    const double lc = fmin(fmax(ln_chi, T.ln_min), T.ln_max);
    const double t = (lc - T.ln_min) * T.inv_delta;
    int k = (int)t;
    k = min(k, T.n_chi - 2);
    *k_out = k;
    *w_out = t - (double)k;
}

// ---- the search of eq.25 / eq.29 -------------------------------------------------------
// Finds m* = max{m : ell(m) <= key} for the row interpolated between rows k and k+1 with weight w
// (eq.24 / eq.28), clamped to M-2, and returns it with a = ell(m*), b = ell(m*+1); -1 when key < ell(0)
// (a photon-emission draw below the first column, R6; P_BW(0) = 0 never is).  The result is the one a plain bisection over [0, M-1] gives (ell is non-decreasing);
// only the schedule differs, because an event is a chain of dependent L2 accesses and its length is what
// costs time: (1) the per-row guide gives a bracket [lo, hi] that provably contains m* (each of the two
// rows bounds the interpolated row); it is verified against the table and dropped if a rounding of the bin
// index made it wrong; (2) a bracket of up to kGuideFastSpan columns (nearly all, with 2048 key bins per row) is
// fetched whole -- ends and interior -- in one round trip and counted; (3) a wider one closes level by level, every
// level probing eight interior points at once (nine-way split): one or two round trips instead of log2(M).
// The guide entries of a key (four 16-bit loads that depend on the row and the key only: the callers issue them together
// with whatever else they load first, one round trip instead of two).
struct GuideBracket { int lo, hi; bool guided; };
constexpr int kGuideFastSpan = 5;   // brackets up to this wide are closed in one round trip (search_row); measured 8 -> 5 -> 4: config 3 event pass 0.0685 -> 0.0669 -> 0.0655 ms, config 5 1.568 -> 1.556 -> 1.558 ms
template <typename R>
__device__ __forceinline__ GuideBracket guide_bracket(const Table2D<R>& T, int k, double key, double r = 0.0) {
    GuideBracket g;
    g.lo = 0;
    g.hi = T.n_xi - 1;
    g.guided = T.guide != nullptr;
    if (g.guided) {
        const int J = T.guide_bins;
        int j = (int)((key - T.guide_k0) * T.guide_inv_dk);
        if (T.guide_split) {   // (key = ln r; the bins above J/2 are uniform in r itself)
            j = min(j, J / 2 - 1);
            if (r >= 0.5) j = J / 2 + (int)((r - 0.5) * (double)J);
        }
        j = max(0, min(j, J - 1));
        const unsigned short* g0 = T.guide + (size_t)k * (J + 1) + j;
        const unsigned short* g1 = g0 + (J + 1);
        const int a0 = __ldg(g0), a1 = __ldg(g0 + 1), b0 = __ldg(g1), b1 = __ldg(g1 + 1);
        g.lo = j == 0 ? 0 : min(a0, b0);
        g.hi = min(max(a1, b1) + 1, T.n_xi - 1);
    }
    return g;
}

template <typename R>
__device__ __forceinline__ int search_row(const Table2D<R>& T, int k, double w, double key, const GuideBracket& gb,
                                          double* a_out, double* b_out) {
    const int M = T.n_xi;
    const R* __restrict__ r0 = T.P + (size_t)k * M;
    const R* __restrict__ r1 = r0 + M;
    auto ell = [&](int m) { const double a = (double)__ldg(r0 + m); return fma(w, (double)__ldg(r1 + m) - a, a); };
    int lo = gb.lo, hi = gb.hi;
    if (gb.guided && hi - lo >= 1 && hi - lo <= kGuideFastSpan) {
        // the common case (99 % of the events with the 2048-bin guide): the bracket is a few columns wide, so its ends
        // (the verification) and its interior are fetched in ONE round trip and counted.
        const int span = hi - lo;
        double v[kGuideFastSpan + 1];
#pragma unroll
        for (int q = 0; q <= kGuideFastSpan; ++q) v[q] = q <= span ? ell(lo + q) : 0.0;
        int cnt = 0;
        bool top_le = false;
#pragma unroll
        for (int q = 1; q <= kGuideFastSpan; ++q) {
            const bool le = q <= span && v[q] <= key;
            cnt += le ? 1 : 0;
            if (q == span) top_le = le;
        }
        if (v[0] <= key && (!top_le || hi == M - 1)) {
            if (cnt == span) --cnt;   // key at or above the last column (only with hi == M-1): the last interval
            double a = v[0], b = v[1];
#pragma unroll
            for (int q = 1; q < kGuideFastSpan; ++q)
                if (q == cnt) { a = v[q]; b = v[q + 1]; }
            *a_out = a;
            *b_out = b;
            return lo + cnt;
        }
        if (lo == 0 && !(v[0] <= key)) return -1;   // key below the first column
        lo = 0;                   // the bracket does not hold (a rounding of the bin index): the full range
        hi = M - 1;
    }
    bool verified = !gb.guided || hi - lo == M - 1;
    bool have_vb = false;         // vb = ell(hi) is known (always, once a guide bracket has been verified)
    double va = 0.0, vb = 0.0;
    if (verified) {               // (unguided: hi = M-1, whose value is fetched at the end if it is still the upper end)
        va = ell(0);
        if (!(va <= key)) return -1;
    }
    while (true) {
        const int span = hi - lo;
        if (verified && span <= 1) break;   // (closed: no probe left to make)
        const int step = (span + 8) / 9;
        double v[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int m = lo + (q + 1) * step;
            v[q] = m < hi ? ell(m) : 0.0;
        }
        if (!verified) {
            va = ell(lo);
            vb = ell(hi);
            verified = true;
            have_vb = true;
            if (!(va <= key) || !(vb > key || hi == M - 1)) {  // guide bracket does not hold: full range
                if (lo == 0 && !(va <= key)) return -1;
                lo = 0;
                hi = M - 1;
                va = ell(0);
                if (!(va <= key)) return -1;
                have_vb = false;
                continue;
            }
        }
        if (span <= 1) break;
        int cnt = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) cnt += (lo + (q + 1) * step < hi && v[q] <= key) ? 1 : 0;
        const int nlo = lo + cnt * step;
        const int nhi_c = lo + (cnt + 1) * step;
        double na = va, nb = vb;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            if (q + 1 == cnt) na = v[q];
            if (q == cnt && nhi_c < hi) nb = v[q];
        }
        if (nhi_c < hi) { hi = nhi_c; have_vb = true; }
        lo = nlo;
        va = na;
        vb = nb;
    }
    if (hi - lo < 1) {            // lo == hi == M-1 (key at or above the last column)
        lo = M - 2;
        va = ell(lo);
        vb = ell(lo + 1);
    } else if (!have_vb) {
        vb = ell(hi);             // the upper end was never probed
    }
    *a_out = va;
    *b_out = vb;
    return lo;
}

// eqs.28-30: xi = chi_gamma/chi of the emitted photon for uniform r (lr = ln r, both passed).
// Event arithmetic is fp64 whatever the table element type (events are rare).
template <typename R>
__device__ __forceinline__ double qs_sample_xi_ln(const Table2D<R>& T, double ln_chi, double lr, double r) {
    int k; double w;
    row_bracket(T, ln_chi, &k, &w);
    const GuideBracket gb = guide_bracket(T, k, lr, r);
    double a, b;
    const int ms = search_row(T, k, w, lr, gb, &a, &b);        // eq.29
    if (ms < 0) return exp_fast(T.ln_xi_min);                  // below the first column (R6)
    const double step = T.xi_step;                             // ln xi_{m+1} - ln xi_m
    const double lx0 = T.ln_xi_min + step * (double)ms;
    if (!(b > a)) return exp_fast(lx0);
    return exp_fast(fma((lr - a) * rcp_fast(b - a), step, lx0));   // eq.30
}
template <typename R>
__device__ __forceinline__ double qs_sample_xi(const Table2D<R>& T, double ln_chi, double r) {
    return qs_sample_xi_ln(T, ln_chi, log_pos(r), r);
}

// eqs.24-26 on r' = min(r, 1-r): xi = chi_-/chi_gamma in [0, 1/2]
template <typename R>
__device__ __forceinline__ double bw_sample_xi(const Table2D<R>& T, double ln_chi, double rp) {
    int k; double w;
    row_bracket(T, ln_chi, &k, &w);
    const int M = T.n_xi;
    double a, b;
    const GuideBracket gb = guide_bracket(T, k, rp);
    const int ms = search_row(T, k, w, rp, gb, &a, &b);        // eq.25 (P(0) = 0 <= r')
    const double step = T.xi_step;
    const double x0 = step * (double)ms;
    if (!(b > a)) return x0;
    return fma((rp - a) * rcp_fast(b - a), step, x0);          // eq.26
}

// ---- 128-bit streaming loads / stores with L2 eviction policies -------------------------------
// The particle arrays are read once per step: they go through L2 as evict-first, so that what is re-used
// (the CDF tables, the guides, the staged records) stays resident in the 126 MB L2.
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long l2_policy_evict_last() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

template <typename T, int V> struct alignas(sizeof(T) * V) Vec { T v[V]; };

// read-only streaming load (never written during the kernel)
template <typename T, int V>
__device__ __forceinline__ Vec<T, V> ld_stream(const T* p, unsigned long long policy) {
    static_assert(sizeof(T) * V == 16, "128-bit vectors");
    Vec<T, V> r;
    uint32_t a, b, c, d;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "l"(p), "l"(policy));
    uint32_t* o = reinterpret_cast<uint32_t*>(&r);
    o[0] = a; o[1] = b; o[2] = c; o[3] = d;
    return r;
}
// the same without .nc, for arrays the kernel also writes (tau)
template <typename T, int V>
__device__ __forceinline__ Vec<T, V> ld_stream_rw(const T* p, unsigned long long policy) {
    static_assert(sizeof(T) * V == 16 || sizeof(T) * V == 32, "128- or 256-bit vectors");
    Vec<T, V> r;
    uint32_t* o = reinterpret_cast<uint32_t*>(&r);
#pragma unroll
    for (int h = 0; h < (int)(sizeof(T) * V / 16); ++h) {
        uint32_t a, b, c, d;
        asm volatile("ld.global.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                     : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "l"(reinterpret_cast<const char*>(p) + 16 * h), "l"(policy) : "memory");
        o[4 * h] = a; o[4 * h + 1] = b; o[4 * h + 2] = c; o[4 * h + 3] = d;
    }
    return r;
}
// plain 128-bit loads that bypass L1 and carry no eviction hint (arrays the fused step rewrites a few microseconds
// later: they should outlive the evict-first field lines in L2)
template <typename T, int V>
__device__ __forceinline__ Vec<T, V> ld_keep(const T* p) {
    static_assert(sizeof(T) * V == 16 || sizeof(T) * V == 32, "128- or 256-bit vectors");
    Vec<T, V> r;
    uint32_t* o = reinterpret_cast<uint32_t*>(&r);
#pragma unroll
    for (int h = 0; h < (int)(sizeof(T) * V / 16); ++h) {
        uint32_t a, b, c, d;
        asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "l"(reinterpret_cast<const char*>(p) + 16 * h) : "memory");
        o[4 * h] = a; o[4 * h + 1] = b; o[4 * h + 2] = c; o[4 * h + 3] = d;
    }
    return r;
}
// vector store in 128-bit pieces: the ABI promises 16-byte alignment only, and a Vec<double, 4> (fp32 particles with an
// fp64 optical depth) stored whole would be one 256-bit store that faults on a 16-byte-aligned view
template <typename T, int V>
__device__ __forceinline__ void st_vec(T* p, const Vec<T, V>& v) {
    static_assert(sizeof(T) * V == 16 || sizeof(T) * V == 32, "128- or 256-bit vectors");
    const uint4* s = reinterpret_cast<const uint4*>(&v);
#pragma unroll
    for (int h = 0; h < (int)(sizeof(T) * V / 16); ++h) reinterpret_cast<uint4*>(p)[h] = s[h];
}
__device__ __forceinline__ void st_policy(uint4* p, const uint4& v, unsigned long long policy) {
    asm volatile("st.global.L2::cache_hint.v4.u32 [%0], {%1,%2,%3,%4}, %5;"
                 ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(policy) : "memory");
}

}  // namespace pxq
