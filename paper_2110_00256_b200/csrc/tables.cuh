// =====================================================================================
//  tables.cuh -- data-parallel GPU builder of the four lookup tables.
//
//  Definitions (PAPER.md:90-110 eqs.4-9, :122 eq.11, :135-162 eqs.12-18):
//     f_BW(chi, xi) = IK_{1/3}(z) + (1/(xi(1-xi)) - 2) K_{2/3}(z),  z = 2/(3 chi xi (1-xi))
//     T(chi) = 1/(pi sqrt3 chi) int_0^1 f_BW dxi,   P_BW(chi, xi) = int_0^xi f_BW / int_0^1 f_BW
//     S/xi = sqrt3/(2 pi) [ IK_{5/3}(Y) + xi^2/(1-xi) K_{2/3}(Y) ],  Y = 2 xi/(3 chi (1-xi))
//     G(chi) = int_0^1 S/xi dxi,                    P_QS(chi, xi) = int_0^xi S/u du / G
//  with K_nu the modified Bessel function and IK_nu(x) = int_x^inf K_nu.
//
//  Numerics (all fp64; different from the CPU oracle's adaptive Gauss-Kronrod on purpose):
//   * K_nu and IK_nu from DLMF 10.32.9, e^x K_nu(x) = int_0^inf exp(-2x sinh^2(t/2)) cosh(nu t) dt,
//     by the trapezoid rule (geometric convergence for this integrand), step
//     h = min(0.25, 0.7/sqrt(x)), hyperbolic functions by addition recurrences;
//   * each table cell [xi_{m-1}, xi_m] is split into panels over which the integrand varies
//     by a bounded factor (rules below) and every panel gets an 8-point Gauss-Legendre rule,
//     one node per lane of an 8-lane group; a CTA owns one table row and turns the cell
//     integrals into the cumulative row with a block scan (rows are monotone by construction);
//   * everything Breit-Wheeler carries the factor e^{z0}, z0 = 8/(3 chi), so that chi down
//     to 1e-4 (ln T ~ -26668) does not underflow (R9).
// =====================================================================================
#pragma once
#include "qed_device.cuh"

namespace pxq {

constexpr int kTabThreads = 256;
constexpr int kTabGroups = kTabThreads / 8;

// 8-point Gauss-Legendre on [-1, 1] (abscissae +-x_k, weights w_k)
__device__ __constant__ double kGL8x[4] = {0.1834346424956498049394761, 0.5255324099163289858177390,
                                           0.7966664774136267395915539, 0.9602898564975362316835609};
__device__ __constant__ double kGL8w[4] = {0.3626837833783619829651504, 0.3137066458778872873379622,
                                           0.2223810344533744705443560, 0.1012285362903762591525314};

// e^z [ cA IK_nuA(z) + cB K_nuB(z) ] = int_0^inf exp(-2 z sinh^2(t/2)) [ cA cosh(nuA t)/cosh t + cB cosh(nuB t) ] dt
__device__ __forceinline__ double bessel_combo_scaled(double z, double nuA, double cA, double nuB, double cB) {
    const double h = fmin(0.25, 0.7 * rsqrt(z));
    const double a = 0.5 * h;
    const double sa = sinh(a), ca = cosh(a);
    const double sA = sinh(nuA * h), cAh = cosh(nuA * h), sB = sinh(nuB * h), cBh = cosh(nuB * h);
    double S = 0.0, C = 1.0;      // sinh(j a), cosh(j a)
    double SA = 0.0, CA = 1.0;    // sinh(j nuA h), cosh(j nuA h)
    double SB = 0.0, CB = 1.0;
    double sum = 0.5 * (cA + cB);
    const double z2 = 2.0 * z;
    for (int j = 1; j < 4096; ++j) {
        const double Sn = fma(S, ca, C * sa);
        C = fma(C, ca, S * sa);
        S = Sn;
        const double SAn = fma(SA, cAh, CA * sA);
        CA = fma(CA, cAh, SA * sA);
        SA = SAn;
        const double SBn = fma(SB, cBh, CB * sB);
        CB = fma(CB, cBh, SB * sB);
        SB = SBn;
        const double s2 = S * S;
        const double ex = z2 * s2;
        if (ex > 46.0) break;
        const double cosht = fma(2.0, s2, 1.0);
        // (the lean reciprocal of qed_device.cuh instead of a division.  The library exp stays: the kernel is bound by the
        // FP64 pipe, and the lean exp_fast, with fewer instructions but more of them FP64, was measured 6 % slower here)
        sum += exp(-ex) * fma(cA * CA, rcp_fast(cosht), cB * CB);
    }
    return sum * h;
}

// ---- Breit-Wheeler ---------------------------------------------------------------------
// With v = 1/(4 xi (1-xi)) >= 1 and y = v - 1 = (1-2 xi)^2/(4 xi (1-xi)):  z = z0 v,  z - z0 = z0 y.
// Integration variable w = sqrt(z0 y): e^{z0} f_BW dxi = e^{-w^2} B(z0 v) (1/2) z0^{-1/2} v^{-3/2} dw,
// B(z) = e^z [IK_{1/3}(z) + (4v - 2) K_{2/3}(z)]: a Gaussian times a smooth function, no singularity at xi = 1/2.
__device__ __forceinline__ double bw_integrand_w(double w, double z0, double inv_sqrt_z0) {
    const double v = fma(w * w, 1.0 / z0, 1.0);
    const double B = bessel_combo_scaled(z0 * v, 1.0 / 3.0, 1.0, 2.0 / 3.0, fma(4.0, v, -2.0));
    return exp(-w * w) * B * 0.5 * inv_sqrt_z0 * rsqrt(v) * rcp_fast(v);
}
__device__ __forceinline__ double bw_y_of_xi(double xi) {
    const double s = 1.0 - 2.0 * xi;
    return s * s / (4.0 * xi * (1.0 - xi));
}

// int over cell [xi_lo, xi_hi] (xi_hi <= 1/2) of e^{z0} f_BW dxi; the 8 lanes of a group each return
// their share (sum over the group = the integral).  Panels: w^2 advances by at most 2 (one e-fold pair
// of the Gaussian) and v at most doubles; the cell is cut where the integrand is e^-44 of its maximum.
__device__ __forceinline__ double bw_cell_share(double chi, double xi_lo, double xi_hi, int node) {
    const double z0 = 8.0 / (3.0 * chi);
    const double inv_sqrt_z0 = rsqrt(z0);
    const double y_a = bw_y_of_xi(xi_hi);
    if (z0 * y_a > 745.0) return 0.0;  // e^{-(z - z0)} underflows: the cell is exactly 0 relative to the row
    const double y_b = xi_lo > 0.0 ? bw_y_of_xi(xi_lo) : INFINITY;
    const double y_end = fmin(y_b, y_a + 44.0 / z0);
    const double gx = (node & 1) ? kGL8x[node >> 1] : -kGL8x[node >> 1];
    const double gw = kGL8w[node >> 1];
    double acc = 0.0;
    double y = y_a;
    while (y < y_end) {
        const double y_next = fmin(fmin(y + 2.0 / z0, fma(2.0, y, 1.0)), y_end);
        if (!(y_next > y)) break;
        const double w0 = sqrt(z0 * y), w1 = sqrt(z0 * y_next);
        const double half = 0.5 * (w1 - w0), mid = 0.5 * (w1 + w0);
        acc = fma(gw * half, bw_integrand_w(fma(half, gx, mid), z0, inv_sqrt_z0), acc);
        y = y_next;
    }
    return acc;
}

// ---- photon emission (QS) --------------------------------------------------------------
// integrand in x = ln xi:  xi * S/xi = xi sqrt3/(2 pi) e^{-Y} e^{Y}[IK_{5/3}(Y) + xi^2/(1-xi) K_{2/3}(Y)]
__device__ __forceinline__ double qs_s_over_xi(double chi, double xi, double one_minus_xi) {
    const double Y = 2.0 * xi / (3.0 * chi * one_minus_xi);
    const double e = exp(-Y);
    if (e == 0.0) return 0.0;
    return 0.2756644477108960 * e * bessel_combo_scaled(Y, 5.0 / 3.0, 1.0, 2.0 / 3.0, xi * xi / one_minus_xi);  // sqrt3/(2 pi)
}

// int over [xi_lo, xi_hi] (0 < xi_lo < xi_hi <= 1) of S/xi dxi, shared over the 8 lanes of a group.
// Panels in x = ln xi: xi grows by at most e^0.6, (1 - xi) at most halves, Y advances by at most 2;
// cut where e^{-Y} has dropped by e^-44 from the start of the cell.
__device__ __forceinline__ double qs_cell_share(double chi, double xi_lo, double xi_hi, int node) {
    const double k = 1.5 * chi;  // Y = xi / (k (1 - xi));  xi = k Y / (1 + k Y)
    const double Y_a = xi_lo / (k * (1.0 - xi_lo));
    if (Y_a > 745.0) return 0.0;       // e^{-Y} underflows
    const double Y_cut = Y_a + 44.0;
    const double xi_end = fmin(xi_hi, k * Y_cut / (1.0 + k * Y_cut));
    const double gx = (node & 1) ? kGL8x[node >> 1] : -kGL8x[node >> 1];
    const double gw = kGL8w[node >> 1];
    double acc = 0.0;
    double xi = xi_lo;
    while (xi < xi_end) {
        const double Y = xi / (k * (1.0 - xi));
        const double Yn = Y + 2.0;
        double xi_next = fmin(xi * 1.8221188003905089, 0.5 * (1.0 + xi));   // e^0.6; (1-xi) halves
        xi_next = fmin(fmin(xi_next, k * Yn / (1.0 + k * Yn)), xi_end);
        if (!(xi_next > xi)) break;
        const double x0 = log(xi), x1 = log(xi_next);
        const double half = 0.5 * (x1 - x0), mid = 0.5 * (x1 + x0);
        const double x = fma(half, gx, mid);
        const double xin = exp(x);
        acc = fma(gw * half, xin * qs_s_over_xi(chi, xin, -expm1(x)), acc);
        xi = xi_next;
    }
    return acc;
}

// int_0^{xi_hi} S/xi dxi: the integrable xi^{-2/3} singularity is removed by xi = v^3 on [0, xi_1],
// xi_1 = min(xi_hi, xi(Y = 1/2)) (two panels); the remainder, if any, goes through qs_cell_share.
__device__ __forceinline__ double qs_first_cell_share(double chi, double xi_hi, int node) {
    const double k = 1.5 * chi;
    const double xi_1 = fmin(xi_hi, 0.5 * k / (1.0 + 0.5 * k));
    const double v1 = cbrt(xi_1);
    const double gx = (node & 1) ? kGL8x[node >> 1] : -kGL8x[node >> 1];
    const double gw = kGL8w[node >> 1];
    double acc = 0.0;
#pragma unroll 1
    for (int p = 0; p < 2; ++p) {
        const double half = 0.25 * v1, mid = (0.25 + 0.5 * p) * v1;
        const double v = fma(half, gx, mid);
        const double xi = v * v * v;
        acc = fma(gw * half, 3.0 * v * v * qs_s_over_xi(chi, xi, 1.0 - xi), acc);
    }
    if (xi_1 < xi_hi) acc += qs_cell_share(chi, xi_1, xi_hi, node);
    return acc;
}

// ---- one CTA per table row ---------------------------------------------------------------
struct TableBuildArgs {
    double chi_min, chi_max;
    int n_chi, n_xi;
    double xi_min;   // QS only
    double* rows;    // n_chi * n_xi: ln P_QS or P_BW (NULL: only the 1D values are wanted)
    double* ln1d;    // n_chi: ln G or ln T (NULL: only the rows are wanted)
};

__device__ __forceinline__ double log_grid(double vmin, double vmax, int n, int i) {
    if (i == 0) return vmin;
    if (i == n - 1) return vmax;
    const double l0 = log(vmin), l1 = log(vmax);
    return exp(l0 + (l1 - l0) * (double)i / (double)(n - 1));
}

template <int KIND>  // 0: photon emission (QS), 1: Breit-Wheeler
__global__ void __launch_bounds__(kTabThreads, 3) table_rows_kernel(const TableBuildArgs a) {
    extern __shared__ double cell[];  // n_xi cell integrals, then the cumulative row
    __shared__ double warp_tot[kTabThreads / 32];
    const int row = blockIdx.x, M = a.n_xi;
    const int tid = threadIdx.x, group = tid >> 3, node = tid & 7, lane = tid & 31, warp = tid >> 5;
    const double chi = log_grid(a.chi_min, a.chi_max, a.n_chi, row);

    // 1. cell integrals: cell m covers [xi_{m-1}, xi_m]; QS cell 0 = [0, xi_min]; BW cell 0 is empty
    for (int m0 = 0; m0 < M; m0 += kTabGroups) {
        const int m = m0 + group;
        double share = 0.0;
        if (m < M) {
            if (KIND == 0) {
                const double hi = log_grid(a.xi_min, 1.0, M, m);
                share = m == 0 ? qs_first_cell_share(chi, hi, node)
                               : qs_cell_share(chi, log_grid(a.xi_min, 1.0, M, m - 1), hi, node);
            } else if (m > 0) {
                const double step = 0.5 / (double)(M - 1);
                share = bw_cell_share(chi, step * (double)(m - 1), m == M - 1 ? 0.5 : step * (double)m, node);
            }
        }
        share += __shfl_xor_sync(0xffffffffu, share, 1);
        share += __shfl_xor_sync(0xffffffffu, share, 2);
        share += __shfl_xor_sync(0xffffffffu, share, 4);
        if (node == 0 && m < M) cell[m] = share;
    }
    __syncthreads();

    // 2. running sum along the row (every term >= 0: the row is monotone by construction, R10)
    const int per = (M + kTabThreads - 1) / kTabThreads;
    const int lo = min(tid * per, M), hi = min(lo + per, M);
    double s = 0.0;
    for (int m = lo; m < hi; ++m) s += cell[m];
    double incl = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const double o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    // exclusive prefix by shifting, never by subtracting: the terms span hundreds of orders of magnitude
    double run = __shfl_up_sync(0xffffffffu, incl, 1);
    if (lane == 0) run = 0.0;
    double before = 0.0;
    for (int w = 0; w < warp; ++w) before += warp_tot[w];
    run += before;
    for (int m = lo; m < hi; ++m) { run += cell[m]; cell[m] = run; }
    __syncthreads();

    // 3. normalise; a prefix maximum removes the last-ulp wiggles of log() and of the division, so that
    //    the stored rows are non-decreasing exactly; store
    const double last = cell[M - 1];
    const double total = KIND == 0 ? last : 2.0 * last;  // BW: f(xi) = f(1 - xi)
    __syncthreads();
    double pm = -INFINITY;
    for (int m = lo; m < hi; ++m) {
        double v;
        if (KIND == 0) v = m == M - 1 ? 0.0 : fmin(log(cell[m] / total), 0.0);  // ln P
        else v = m == 0 ? 0.0 : (m == M - 1 ? 0.5 : fmin(cell[m] / total, 0.5));
        pm = fmax(pm, v);
        cell[m] = pm;
    }
    double wm = pm;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) wm = fmax(wm, __shfl_up_sync(0xffffffffu, wm, d));
    // (lanes < d read their own value back from shfl_up, so the max is unchanged for them)
    __syncthreads();
    if (lane == 31) warp_tot[warp] = wm;
    __syncthreads();
    double floor_v = __shfl_up_sync(0xffffffffu, wm, 1);
    if (lane == 0) floor_v = -INFINITY;
    for (int w = 0; w < warp; ++w) floor_v = fmax(floor_v, warp_tot[w]);
    if (a.rows != nullptr) {
        double* out = a.rows + (size_t)row * M;
        for (int m = lo; m < hi; ++m) out[m] = fmax(cell[m], floor_v);
    }
    if (tid == 0 && a.ln1d != nullptr) {
        if (KIND == 0) a.ln1d[row] = log(total);                                             // ln G
        else a.ln1d[row] = log(total / (kPi * 1.7320508075688772 * chi)) - 8.0 / (3.0 * chi);  // ln T (eq.9)
    }
}

}  // namespace pxq
