// =====================================================================================
//  cascade.cuh -- the closed loop in a uniform field:
//  what surrounds the QED step when secondaries are fed back.
//    boris_kernel        leptons pushed in uniform e, b (R19)                       HBM, 48/24 B per particle
//    keep_count_kernel   \  ordered, filtering append of the new secondaries to a species'
//    append_kernel       /  arrays: photons below the energy threshold are discarded at
//                           creation (R22); order is kept (ballot/popc + the
//                           block scan of events.cuh)
//    spectrum_kernel     energy histogram over logarithmic bins (Fig.6, R23)                   HBM, 24/12 B per particle
//    fill_kernel         constant field arrays for the QED step
// =====================================================================================
#pragma once
#include "qed_device.cuh"
#include "evolve.cuh"

namespace pxq {

constexpr double kInvTauC = kElectronMass * kLightSpeed * kLightSpeed / (kPlanck / (2.0 * kPi));  // m c^2/hbar, 1/s

// ---- classical radiation reaction below the chi threshold (R24) ---------------------------------
// A lepton with chi < chi_min loses kinetic energy at the classical radiated power, the chi -> 0 limit of the mean loss of
// the Monte Carlo emission: d(gamma-1)/dt = -(2/3)(alpha/tau_C) chi^2 (gamma-1)/gamma; direction kept, norm(p') from gamma'.
// One streaming pass: nine 128-bit loads per thread, chi^2 in fp64 registers (the routine of the evolve pass), and the three
// momentum vectors stored back only where a lepton of the vector was below the threshold.
template <typename R>
__global__ void __launch_bounds__(256) classical_loss_kernel(R* __restrict__ px, R* __restrict__ py, R* __restrict__ pz,
                                                             const R* __restrict__ ex, const R* __restrict__ ey,
                                                             const R* __restrict__ ez, const R* __restrict__ bx,
                                                             const R* __restrict__ by, const R* __restrict__ bz, long long n,
                                                             double c2_min, double loss_dt /* (2/3)(alpha/tau_C) dt */) {
    constexpr int V = 16 / sizeof(R);
    const long long nvec = n / V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const unsigned long long pol = l2_policy_evict_first();
    auto one = [&](R& x, R& y, R& z, R e0, R e1, R e2, R b0, R b1, R b2) -> bool {
        double inv_g, g2;
        const double c2 = chi_squared_of<0>(x, y, z, e0, e1, e2, b0, b1, b2, &inv_g, &g2);
        const double p2 = g2 - 1.0;
        if (!(c2 < c2_min) || !(p2 > 1e-300)) return false;
        const double g = g2 * inv_g;
        const double k = p2 * rcp_fast(g + 1.0);                       // gamma - 1
        double k2 = k - loss_dt * c2 * (k * inv_g);
        k2 = k2 > 0.0 ? k2 : 0.0;
        const double q2 = k2 * (k2 + 2.0);
        const double s = q2 > 1e-300 ? q2 * rsqrt_fast(q2) * rsqrt_fast(p2) : 0.0;
        x = (R)(s * x); y = (R)(s * y); z = (R)(s * z);
        return true;
    };
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < nvec; j += stride) {
        const long long i = j * V;
        Vec<R, V> x = ld_stream_rw<R, V>(px + i, pol), y = ld_stream_rw<R, V>(py + i, pol), z = ld_stream_rw<R, V>(pz + i, pol);
        const Vec<R, V> a3 = ld_stream<R, V>(ex + i, pol), a4 = ld_stream<R, V>(ey + i, pol), a5 = ld_stream<R, V>(ez + i, pol),
                        a6 = ld_stream<R, V>(bx + i, pol), a7 = ld_stream<R, V>(by + i, pol), a8 = ld_stream<R, V>(bz + i, pol);
        bool any = false;
#pragma unroll
        for (int v = 0; v < V; ++v) any = one(x.v[v], y.v[v], z.v[v], a3.v[v], a4.v[v], a5.v[v], a6.v[v], a7.v[v], a8.v[v]) || any;
        if (any) {
            st_vec<R, V>(px + i, x);
            st_vec<R, V>(py + i, y);
            st_vec<R, V>(pz + i, z);
        }
    }
    for (long long i = nvec * V + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        R x = px[i], y = py[i], z = pz[i];
        if (one(x, y, z, ex[i], ey[i], ez[i], bx[i], by[i], bz[i])) { px[i] = x; py[i] = y; pz[i] = z; }
    }
}

// ---- Boris push in a uniform field (R19) ---------------------------------------------------------------
// ke = s dt/(2 tau_C) e, kb = s dt/(2 tau_C) b (host, fp64).  Arithmetic in fp64 registers whatever R.
struct BorisArgs {
    double ke[3], kb[3];
};

__device__ __forceinline__ void boris_one(double& ux, double& uy, double& uz, const BorisArgs& a) {
    const double mx = ux + a.ke[0], my = uy + a.ke[1], mz = uz + a.ke[2];            // half electric kick
    const double inv_g = rsqrt_fast(1.0 + fma(mx, mx, fma(my, my, mz * mz)));        // 1/gamma^-
    const double tx = a.kb[0] * inv_g, ty = a.kb[1] * inv_g, tz = a.kb[2] * inv_g;    // rotation vector
    const double px = mx + (my * tz - mz * ty);                                       // u' = u^- + u^- x t
    const double py = my + (mz * tx - mx * tz);
    const double pz = mz + (mx * ty - my * tx);
    const double f = 2.0 * rcp_fast(1.0 + fma(tx, tx, fma(ty, ty, tz * tz)));
    const double sx = f * tx, sy = f * ty, sz = f * tz;
    ux = mx + (py * sz - pz * sy) + a.ke[0];                                          // u^+ = u^- + u' x s, second half kick
    uy = my + (pz * sx - px * sz) + a.ke[1];
    uz = mz + (px * sy - py * sx) + a.ke[2];
}

template <typename R>
__global__ void __launch_bounds__(256) boris_kernel(R* __restrict__ px, R* __restrict__ py, R* __restrict__ pz, long long n,
                                                    const BorisArgs a) {
    constexpr int V = 16 / sizeof(R);
    const long long nvec = n / V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const unsigned long long pol = l2_policy_evict_first();
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < nvec; j += stride) {
        Vec<R, V> x = ld_stream_rw<R, V>(px + j * V, pol), y = ld_stream_rw<R, V>(py + j * V, pol),
                  z = ld_stream_rw<R, V>(pz + j * V, pol);
#pragma unroll
        for (int v = 0; v < V; ++v) {
            double ux = x.v[v], uy = y.v[v], uz = z.v[v];
            boris_one(ux, uy, uz, a);
            x.v[v] = (R)ux; y.v[v] = (R)uy; z.v[v] = (R)uz;
        }
        *reinterpret_cast<Vec<R, V>*>(px + j * V) = x;
        *reinterpret_cast<Vec<R, V>*>(py + j * V) = y;
        *reinterpret_cast<Vec<R, V>*>(pz + j * V) = z;
    }
    for (long long i = nvec * V + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        double ux = px[i], uy = py[i], uz = pz[i];
        boris_one(ux, uy, uz, a);
        px[i] = (R)ux; py[i] = (R)uy; pz[i] = (R)uz;
    }
}

// ---- ordered, filtering append (R20, R22) -----------------------------------------------------------
// keep(i) = !(|p_i| < min_energy), |p| = sqrt((px^2 + py^2) + pz^2) with every operation rounded separately
// (no fma): the decision is then the one an fp64 evaluation of the same expression takes anywhere.
template <typename R>
__device__ __forceinline__ bool keep_entry(const R* px, const R* py, const R* pz, long long i, double min_energy) {
    const double x = px[i], y = py[i], z = pz[i];
    const double g = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z)));
    return !(g < min_energy);
}

// level 1: one warp per 128-entry chunk of the source; m = min(*d_count, m_max) valid entries
template <typename R>
__global__ void __launch_bounds__(256) keep_count_kernel(const R* __restrict__ px, const R* __restrict__ py,
                                                         const R* __restrict__ pz, const unsigned long long* d_count,
                                                         long long m_max, double min_energy, long long n_chunks,
                                                         unsigned short* __restrict__ cnt) {
    const int lane = threadIdx.x & 31;
    const long long m = (long long)min((unsigned long long)m_max, *d_count);
    n_chunks = min(n_chunks, (m + kChunk - 1) / kChunk);   // only the chunks that hold entries (the scan does the same)
    const long long warps = (long long)gridDim.x * (blockDim.x / 32);
    for (long long ch = (long long)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5); ch < n_chunks; ch += warps) {
        unsigned int k = 0;
#pragma unroll
        for (int r4 = 0; r4 < kChunk / 32; ++r4) {
            const long long i = ch * kChunk + r4 * 32 + lane;
            const bool f = i < m && keep_entry(px, py, pz, i, min_energy);
            k += __popc(__ballot_sync(0xffffffffu, f));
        }
        if (lane == 0) cnt[ch] = (unsigned short)k;
    }
}

constexpr int kAppendChunksPerTile = 8;

// level 3 (level 2 is tile_scan_kernel with kAppendChunksPerTile): entry i of the source that is kept goes to
// dst[dst_n + (number of kept entries before i)]; entries past dst_capacity are dropped, *d_new_n = dst_n + kept
// tells (the caller checks it against the capacity)
template <typename R, typename TR>
struct AppendArgs {
    const R* s_p[3];
    const TR* s_tau;
    R* d_p[3];
    TR* d_tau;
    const unsigned long long* d_count;
    long long m_max, dst_n, dst_capacity, n_chunks;
    const unsigned long long* d_dst_n;   // not NULL: the destination starts at *d_dst_n instead of dst_n
    double min_energy;
    const unsigned short* cnt;
    const unsigned long long* tile_offset;
    const unsigned long long* d_kept;
    unsigned long long* d_new_n;
};

template <typename R, typename TR>
__global__ void __launch_bounds__(256) append_kernel(const AppendArgs<R, TR> a) {
    const int lane = threadIdx.x & 31;
    const long long m = (long long)min((unsigned long long)a.m_max, *a.d_count);
    const long long dst_n = a.d_dst_n ? (long long)*a.d_dst_n : a.dst_n;
    if (blockIdx.x == 0 && threadIdx.x == 0) *a.d_new_n = (unsigned long long)dst_n + *a.d_kept;
    const long long warps = (long long)gridDim.x * (blockDim.x / 32);
    const long long n_chunks = min(a.n_chunks, (m + kChunk - 1) / kChunk);
    for (long long ch = (long long)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5); ch < n_chunks; ch += warps) {
        const long long tile = ch / kAppendChunksPerTile;
        const int in_tile = (int)(ch - tile * kAppendChunksPerTile);
        const unsigned int c = lane < in_tile ? a.cnt[tile * kAppendChunksPerTile + lane] : 0u;   // chunks before this one
        long long slot = dst_n + (long long)a.tile_offset[tile] + __reduce_add_sync(0xffffffffu, c);
#pragma unroll
        for (int r4 = 0; r4 < kChunk / 32; ++r4) {
            const long long i = ch * kChunk + r4 * 32 + lane;
            const bool f = i < m && keep_entry(a.s_p[0], a.s_p[1], a.s_p[2], i, a.min_energy);
            const unsigned int bal = __ballot_sync(0xffffffffu, f);
            const long long d = slot + __popc(bal & ((1u << lane) - 1u));
            if (f && d < a.dst_capacity) {
#pragma unroll
                for (int k = 0; k < 3; ++k) a.d_p[k][d] = a.s_p[k][i];
                a.d_tau[d] = a.s_tau[i];
            }
            slot += __popc(bal);
        }
    }
}

// ---- energy spectrum (R23) --------------------------------------------------------------------------
// bin = floor((ln E - ln e_min) * scale), scale = nbins/(ln e_max - ln e_min), in fp64; E = gamma - 1 =
// p^2/(gamma + 1) for leptons, |p| for photons; p = 0 (dead) and out-of-range energies are skipped.
// Shared-memory counters per CTA (nbins <= kSpectrumMaxBins), flushed with one atomic per non-empty bin.
constexpr int kSpectrumMaxBins = 8192;

template <int SPECIES>
__device__ __forceinline__ void spectrum_one(double x, double y, double z, double ln_min, double scale, int nbins,
                                             unsigned int* bins) {
    const double p2 = __dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z));
    if (!(p2 > 0.0)) return;
    const double en = SPECIES == 0 ? p2 / (__dsqrt_rn(1.0 + p2) + 1.0) : __dsqrt_rn(p2);
    const double pos = (log(en) - ln_min) * scale;
    if (pos >= 0.0 && pos < (double)nbins) atomicAdd(&bins[(int)floor(pos)], 1u);
}

template <typename R, int SPECIES>
__global__ void __launch_bounds__(256) spectrum_kernel(const R* __restrict__ px, const R* __restrict__ py,
                                                       const R* __restrict__ pz, long long n, double ln_min, double scale,
                                                       int nbins, unsigned long long* __restrict__ hist) {
    extern __shared__ unsigned int bins[];
    for (int k = threadIdx.x; k < nbins; k += blockDim.x) bins[k] = 0u;
    __syncthreads();
    constexpr int V = 16 / sizeof(R);
    const long long nvec = n / V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const unsigned long long pol = l2_policy_evict_first();
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < nvec; j += 2 * stride) {
        // two 128-bit loads per array per thread in flight
        const long long j2 = j + stride;
        Vec<R, V> x0 = ld_stream<R, V>(px + j * V, pol), y0 = ld_stream<R, V>(py + j * V, pol),
                  z0 = ld_stream<R, V>(pz + j * V, pol);
        Vec<R, V> x1 = x0, y1 = y0, z1 = z0;
        if (j2 < nvec) {
            x1 = ld_stream<R, V>(px + j2 * V, pol);
            y1 = ld_stream<R, V>(py + j2 * V, pol);
            z1 = ld_stream<R, V>(pz + j2 * V, pol);
        }
#pragma unroll
        for (int v = 0; v < V; ++v) spectrum_one<SPECIES>(x0.v[v], y0.v[v], z0.v[v], ln_min, scale, nbins, bins);
        if (j2 < nvec) {
#pragma unroll
            for (int v = 0; v < V; ++v) spectrum_one<SPECIES>(x1.v[v], y1.v[v], z1.v[v], ln_min, scale, nbins, bins);
        }
    }
    for (long long i = nvec * V + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        spectrum_one<SPECIES>(px[i], py[i], pz[i], ln_min, scale, nbins, bins);
    __syncthreads();
    for (int k = threadIdx.x; k < nbins; k += blockDim.x)
        if (bins[k]) atomicAdd(&hist[k], (unsigned long long)bins[k]);
}

template <typename R>
__global__ void __launch_bounds__(256) fill_kernel(R* __restrict__ out, long long n, R value) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) out[i] = value;
}

}  // namespace pxq
