// =====================================================================================
//  lookup.cuh -- the table functions as the hot path evaluates them, exposed per value
//  (the table-accuracy study of PAPER.md Figs.2-5 runs on these).
//    table_function_kernel   G(chi) (eq.27) or T(chi_gamma) (eq.23, Erber form outside the table)
//    sample_xi_kernel        xi(chi, r) by inverse-CDF lookup: eqs.28-30 (photon emission), eqs.24-26 with the
//                            r -> 1 - r reflection of PAPER.md:212 (pair production; xi = chi_-/chi_gamma)
//  Neither kernel has arithmetic of its own: the first runs decrement_one (evolve.cuh) on a synthetic particle whose
//  quantum parameter is chi, the second calls qs_sample_xi / bw_sample_xi (qed_device.cuh), the routines of the
//  event pass.
// =====================================================================================
#pragma once
#include "qed_device.cuh"
#include "evolve.cuh"

namespace pxq {

// A particle with p = (g, 0, 0), e = 0, b = (0, 0, chi/g) has chi^2 = (g b_z)^2 exactly (eq.2 / eq.3 with e = 0);
// with rate_dt = 1 its decrement is G(chi)/gamma (leptons) or chi T(chi)/gamma_gamma (photons).
template <typename R, int KIND>
__global__ void __launch_bounds__(256) table_function_kernel(const R* __restrict__ chi, R* __restrict__ out, long long n,
                                                             const Table1D<R> T) {
    const double g = 1024.0;  // (a power of two: chi/g and g*(chi/g) are exact)
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const double c = chi[i];
        const R d = decrement_one<R, KIND>((R)g, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)0, (R)(c / g), T.L, T, 1.0, UnitScales());
        const double gamma = KIND == 0 ? sqrt(1.0 + g * g) : g;
        out[i] = KIND == 0 ? (R)((double)d * gamma) : (R)((double)d * gamma / c);
    }
}

template <typename R, int KIND>
__global__ void __launch_bounds__(256) sample_xi_kernel(const R* __restrict__ chi, const R* __restrict__ r,
                                                        R* __restrict__ xi, long long n, const Table2D<R> cdf) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const double lc = log((double)chi[i]), u = r[i];
        if (KIND == 0) {
            xi[i] = (R)qs_sample_xi(cdf, lc, u);
        } else {
            const bool electron_side = u <= 0.5;
            const double x = bw_sample_xi(cdf, lc, electron_side ? u : 1.0 - u);
            xi[i] = (R)(electron_side ? x : 1.0 - x);
        }
    }
}

}  // namespace pxq
