// =====================================================================================
//  evolve.cuh -- chi, optical-depth initialisation and the fused
//  chi + 1D-table lookup + optical-depth update kernel.
//
//  Streaming kernels over structure-of-arrays particle buffers: 128-bit loads that bypass
//  L1, the ln G / ln T table staged once per CTA in shared memory by a TMA bulk copy,
//  persistent grid sized to the SM count.  HBM traffic per particle = the ten reals of
//  PAPER.md:301 plus the optical-depth write: 88 B (fp64), 44 B (fp32), 52 B (fp32 + fp64 tau).
// =====================================================================================
#pragma once
#include "qed_device.cuh"

namespace pxq {

constexpr int kEvolveThreads = 256;

template <typename R, typename TR>
struct EvolveArgs {
    const R* p[3];
    const R* e[3];
    const R* b[3];
    TR* tau;
    long long n;
    Table1D<R> tab;
    double rate_dt;            // (2/3) alpha/tau_C dt (leptons) or alpha/tau_C dt (photons)
    unsigned int* partials;    // gridDim.x per-CTA event counts (ctx scratch), or nullptr
    unsigned int* ticket;      // self-resetting arrival counter (ctx scratch)
    unsigned long long* d_n_events;
    int table_in_smem;
    // record emission (EMIT kernels only): every 128-particle chunk owns a segment of kStageCap records
    unsigned char* stage_rec;   // [n_chunks] segments of kStageCap records (see StageRecord), in index order
    long long stage_stride;     // bytes from one chunk's segment to the next
    unsigned short* stage_cnt;  // [n_chunks]: fired particles of the chunk | flags (see kStage* below)
    unsigned table_bytes;       // dynamic shared memory: [table, padded to 128 B][per-warp record buffers]
    // EMIT: every chunk count is also added to the sum of its event tile (one RED per warp and tile), so that the
    // offsets scan reads one word per tile instead of every chunk count
    unsigned int* tile_sum;
    int chunks_per_tile;
    int remove_photons;         // EMIT, photons: 1 = the pass removes the photons it stages (qed_step), 0 = it only stages
    // EMIT, leptons: 1 = the pass also re-draws the optical depth of the leptons it stages (qed_step: tau = -ln U from the parent's
    // Philox words), so that it leaves with the pass's own vector store and the event pass rewrites three scattered
    // sectors per event instead of four; the evolved value stays in the record (capacity rule)
    int redraw_tau;
    unsigned long long seed, step, id_base;
    UnitScales units;           // the caller's unit system (picsarqed_set_units)
};

constexpr int kEventTileChunks = 32;        // chunks per tile of event_kernel (the tile sums are kept per 32 chunks: a shift,
                                            // not a 64-bit division, in the kernels that count)
constexpr int kChunk = 128;                 // particles one warp handles per tile: the unit of record staging
constexpr int kStageCap = 24;               // records per chunk segment (mean at 5 % firing: 6.4)
// stage_cnt[chunk]: bits 0..14 = number of particles of the chunk that fired; bit 15 = the chunk has no staged
// records (segment overflow, or counted by count_chunks_kernel: generate_* calls and the ragged last tile)
// bit 14 = the events of the chunk have been generated already (fused step, step.cuh): its segment holds StepResult
// records -- the secondaries, waiting for their slots
// bit 13 = the evolve pass has done its part of the parents' rewrite already, with its own stores: photons are removed (p = 0,
// tau = +inf: the event pass only creates the pairs), leptons have their new optical depth (the event pass rewrites the momentum only)
constexpr unsigned short kStageCountMask = 0x1FFFu;
constexpr unsigned short kStageNoRecords = 0x8000u;
constexpr unsigned short kStageDone = 0x4000u;
constexpr unsigned short kStageParentDone = 0x2000u;

// one staged record: what event generation needs of a particle that fired -- its momentum, chi^2 (computed by the
// evolve pass anyway) and its index inside the chunk.  Sizes are multiples of 16 bytes so that records move as
// 128-bit vectors.  (Also staging the fields, 80 B, was measured: it made the evolve pass slower by more than the event
// pass gained.  Re-drawing the parent's optical depth in the evolve pass -- compacted into one warp pass per chunk, the
// evolved value kept in the record for the capacity rule -- is what EvolveArgs::redraw_tau does.)
template <typename R> struct StageRecord;
// tau_ev: the evolved optical depth (what undoes a removed photon that falls beyond the capacity of the output)
template <> struct alignas(16) StageRecord<double> {
    double p[3]; double c2; unsigned idx; unsigned pad; double tau_ev;
    static constexpr int kBytes = 48, kVecs = 3;
};
template <> struct alignas(16) StageRecord<float> {
    float p[3]; unsigned idx; double c2; double tau_ev;
    static constexpr int kBytes = 32, kVecs = 2;
};
static_assert(sizeof(StageRecord<double>) == 48 && sizeof(StageRecord<float>) == 32, "record layout");

// one staged result of the fused step (step.cuh): the secondaries of an event whose parent has been rewritten already,
// plus what undoes that rewrite if the event falls beyond the capacity of the output (R16): the parent's old
// momentum, its evolved optical depth and its index in the chunk.  KIND 0: one photon; KIND 1: electron and positron.
template <typename R, typename TR, int KIND> struct alignas(16) StepResult {
    TR sec_tau[KIND == 0 ? 1 : 2];
    TR tau_ev;
    R sec[KIND == 0 ? 3 : 6];
    R old_p[3];
    unsigned idx;
};
static_assert(sizeof(StepResult<double, double, 0>) == 80 && sizeof(StepResult<float, double, 0>) == 48 &&
              sizeof(StepResult<float, float, 0>) == 48 && sizeof(StepResult<double, double, 1>) == 112 &&
              sizeof(StepResult<float, double, 1>) == 64 && sizeof(StepResult<float, float, 1>) == 64, "result layout");

// ---- TMA bulk copy of a 1D table into shared memory ------------------------------------
__device__ __forceinline__ void stage_table_tma(void* smem_dst, const void* gmem_src, unsigned bytes,
                                                unsigned long long* mbar) {
    const unsigned mb = (unsigned)__cvta_generic_to_shared(mbar);
    const unsigned dst = (unsigned)__cvta_generic_to_shared(smem_dst);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst), "l"(gmem_src), "r"(bytes), "r"(mb) : "memory");
    }
    unsigned done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(mb) : "memory");
    }
}

// ---- one particle ----------------------------------------------------------------------
// a_k(1/3) of the Hankel expansion of K_{1/3} (DLMF 10.40.2, 10.17.1): a_k = prod_{j=1..k} (4 nu^2 - (2j-1)^2)/(8 j);
// evaluated by the compiler (the callers pass literals)
__host__ __device__ constexpr double hankel13(int k) {
    double a = 1.0;
    for (int j = 1; j <= k; ++j) a *= (4.0 / 9.0 - (2.0 * j - 1.0) * (2.0 * j - 1.0)) / (8.0 * j);
    return a;
}

// Outside the T table: chi T = 0.16 K_{1/3}(x)^2, x = 4/(3 chi) (eq.10 with the argument of DESIGN.md R2).
// A routine of its own: for fp32 particles it is called (not inlined), so that the registers of the streaming kernel are
// those of its common path (in-table photons) and three CTAs fit on an SM.
template <typename R>
__device__ __forceinline__ R erber_decrement_body(double c2, double inv_g, double rate_dt) {
    typedef R A;
        // chi T = 0.16 K_{1/3}(x)^2, x = 4/(3 chi) (eq.10 with the argument of DESIGN.md R2)
        if (c2 < 1.7777e-4) return (A)0;  // x > 100: K^2 < e^-200, the decrement is below 1e-80 of any optical depth
        if constexpr (sizeof(R) == 4) {
            if (c2 > 7.2e2) {  // x < 0.05, fp32 particles: the same series in float (two terms: y < 7e-4)
                const float y = (4.0f / 9.0f) / (float)c2;
                const float sm = (float)(1.0 / 1.3541179394264004) * fmaf(y, 1.5f, 1.0f);
                const float sp = (float)(1.0 / 0.8929795115692492) * fmaf(y, 0.75f, 1.0f);
                const float h2 = cbrtf(y);
                const float k = sm - sp * h2;
                return (float)rate_dt * (0.16f * 3.2898681336964524f) * (k * k / h2) * (float)inv_g;  // (pi/sqrt3)^2
            }
        }
        double k2;                        // K_{1/3}(x)^2
        if (c2 > 7.2e2) {                 // x < 0.05
            // ascending series (DLMF 10.27.4, 10.25.2), four terms: relative error < (x^2/4)^4 < 2e-13.
            // K = (pi/sqrt3) (sm/h - sp h), h = (x/2)^(1/3); with y = x^2/4 = 4/(9 chi^2): h^2 = cbrt(y)
            // (coefficients 1/(k (k -+ nu)) are written as constants: no divisions in the series)
            const double y = (4.0 / 9.0) / c2;
            constexpr double am1 = 1.0 / (1.0 * (1.0 - 1.0 / 3.0)), am2 = 1.0 / (2.0 * (2.0 - 1.0 / 3.0)),
                             am3 = 1.0 / (3.0 * (3.0 - 1.0 / 3.0));
            constexpr double ap1 = 1.0 / (1.0 * (1.0 + 1.0 / 3.0)), ap2 = 1.0 / (2.0 * (2.0 + 1.0 / 3.0)),
                             ap3 = 1.0 / (3.0 * (3.0 + 1.0 / 3.0));
            const double sm = (1.0 / 1.3541179394264004) * fma(y * am1, fma(y * am2, fma(y, am3, 1.0), 1.0), 1.0);
            const double sp = (1.0 / 0.8929795115692492) * fma(y * ap1, fma(y * ap2, fma(y, ap3, 1.0), 1.0), 1.0);
            const double h2 = cbrt(y);
            const double k = sm - sp * h2;  // K h sqrt3/pi
            k2 = (1.5707963267948966 / 0.8660254037844386) * (1.5707963267948966 / 0.8660254037844386) * k * k / h2;
        } else if (c2 < 2.8444e-3) {      // x > 25: the window just below a T table that starts at chi ~ 1e-2
            // Hankel expansion (DLMF 10.40.2): K^2 = (pi/2x) e^{-2x} (sum_k a_k x^-k)^2, sixteen terms in
            // Horner form with constant coefficients (the first term left out is < 1e-16 at x = 25); 1/x =
            // (3/4) chi comes from one rsqrt: no division, no logarithm
            const double rs = rsqrt_fast(c2);
            const double x = (4.0 / 3.0) * rs, r = 0.75 * (c2 * rs);
            double sum = hankel13(16);
#pragma unroll
            for (int k = 15; k >= 1; --k) sum = fma(sum, r, hankel13(k));
            sum = fma(sum, r, 1.0);
            k2 = 1.5707963267948966 * r * sum * sum * exp_fast(-2.0 * x);
        } else {
            const double x = 4.0 / (3.0 * sqrt(c2));
            k2 = exp(2.0 * (ln_bessel_k13_scaled(x) - x));
        }
        return (A)(rate_dt * 0.16 * k2 * inv_g);
}
__device__ __noinline__ float erber_decrement_f32(double c2, double inv_g, double rate_dt) {
    return erber_decrement_body<float>(c2, inv_g, rate_dt);
}
template <typename R>
__device__ __forceinline__ R erber_decrement(double c2, double inv_g, double rate_dt) {
    if constexpr (sizeof(R) == 4) return erber_decrement_f32(c2, inv_g, rate_dt);
    else return erber_decrement_body<R>(c2, inv_g, rate_dt);
}

// The decrement dN/dt * dt from chi^2 (all cases, one particle), in the particle arithmetic type A = R.
template <typename R, int SPECIES>
__device__ __forceinline__ R rate_from_c2(double c2, double inv_g, double g2, const R* tab, const Table1D<R>& T,
                                          double rate_dt) {
    typedef R A;
    if (c2 < T.c2_event_min) return (A)0;   // below the chi threshold of PAPER.md:340 neither process is an event (R24)
    A lc;
    if constexpr (sizeof(R) == 8) lc = 0.5 * log_pos(c2); else lc = 0.5f * logf((float)c2);
    const A ln_min = (A)T.ln_min, ln_max = (A)T.ln_max, inv_delta = (A)T.inv_delta;
    if (SPECIES == 0) {
        // eq.15 with G from eq.27; first/last value outside the table
        lc = lc < ln_min ? ln_min : (lc > ln_max ? ln_max : lc);
        const A L = lookup_ln<R, A>(tab, T.n, lc, ln_min, inv_delta);
        if constexpr (sizeof(R) == 8) return rate_dt * exp_fast(L) * inv_g;
        else return (float)rate_dt * expf(L) * (float)inv_g;
    } else {
        // eq.8 with T from eq.23; Erber form outside; gamma_gamma <= 2 cannot decay (R12)
        if (!(g2 > 4.0) || !(c2 > 0.0)) return (A)0;
        if (c2 < T.chi_min * T.chi_min || c2 > T.chi_max * T.chi_max) {
            if (c2 < 1.7777e-4) return (A)0;  // (the routine's own first test, kept here: no call for the photons far below)
            return erber_decrement<R>(c2, inv_g, rate_dt);
        }
        lc = lc < ln_min ? ln_min : (lc > ln_max ? ln_max : lc);
        const A L = lookup_ln<R, A>(tab, T.n, lc, ln_min, inv_delta);
        if constexpr (sizeof(R) == 8) return rate_dt * exp_fast(L + lc) * inv_g;
        else return (float)rate_dt * expf(L + lc) * (float)inv_g;
    }
}

// Returns the decrement dN/dt * dt in the particle arithmetic type (float or double).
// SCALED: the arrays are in another unit system (picsarqed_set_units): nine multiplications in registers.
template <typename R, int SPECIES, bool SCALED = false>
__device__ __forceinline__ auto decrement_one(R pxr, R pyr, R pzr, R exr, R eyr, R ezr, R bxr, R byr, R bzr,
                                              const R* tab, const Table1D<R>& T, double rate_dt,
                                              const UnitScales& us, double* c2_out = nullptr) -> R {
    double inv_g, g2;
    const double c2 =
        SCALED ? chi_squared_of<SPECIES>(pxr * us.p, pyr * us.p, pzr * us.p, exr * us.e, eyr * us.e, ezr * us.e,
                                         bxr * us.b, byr * us.b, bzr * us.b, &inv_g, &g2)
               : chi_squared_of<SPECIES>(pxr, pyr, pzr, exr, eyr, ezr, bxr, byr, bzr, &inv_g, &g2);
    if (c2_out) *c2_out = c2;
    return rate_from_c2<R, SPECIES>(c2, inv_g, g2, tab, T, rate_dt);
}

// The same for the V particles a thread holds in one 128-bit vector per array: identical arithmetic, but the common path
// (leptons; photons inside the T table) is written stage by stage over the V particles, so that it is one straight line
// the compiler can interleave, with the logarithm and the exponential in their V-at-once forms (qed_device.cuh).
// in[c][v]: component c (px, py, pz, ex, ey, ez, bx, by, bz) of particle v.
template <typename R, int SPECIES, bool SCALED, int V>
__device__ __forceinline__ void decrement_vec(const R (&in)[9][V], const R* tab, const Table1D<R>& T, double rate_dt,
                                              const UnitScales& us, R (&d)[V], double (&c2)[V]) {
    double inv_g[V], g2[V];
#pragma unroll
    for (int v = 0; v < V; ++v)
        c2[v] = SCALED ? chi_squared_of<SPECIES>(in[0][v] * us.p, in[1][v] * us.p, in[2][v] * us.p, in[3][v] * us.e,
                                                 in[4][v] * us.e, in[5][v] * us.e, in[6][v] * us.b, in[7][v] * us.b,
                                                 in[8][v] * us.b, &inv_g[v], &g2[v])
                       : chi_squared_of<SPECIES>(in[0][v], in[1][v], in[2][v], in[3][v], in[4][v], in[5][v], in[6][v],
                                                 in[7][v], in[8][v], &inv_g[v], &g2[v]);
    if constexpr (sizeof(R) == 8) {
        double lc[V], L[V], ex[V];
        log_pos_v<V>(c2, lc);
        const double ln_min = T.ln_min, ln_max = T.ln_max, inv_delta = T.inv_delta;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            lc[v] = 0.5 * lc[v];
            lc[v] = lc[v] < ln_min ? ln_min : (lc[v] > ln_max ? ln_max : lc[v]);
            L[v] = lookup_ln<R, double>(tab, T.n, lc[v], ln_min, inv_delta);
            if (SPECIES == 1) L[v] = L[v] + lc[v];                                  // eq.8: chi T
        }
        exp_fast_v<V>(L, ex);
#pragma unroll
        for (int v = 0; v < V; ++v) d[v] = c2[v] < T.c2_event_min ? 0.0 : rate_dt * ex[v] * inv_g[v];
    } else {
        const float ln_min = (float)T.ln_min, ln_max = (float)T.ln_max, inv_delta = (float)T.inv_delta;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            float lc = 0.5f * logf((float)c2[v]);
            lc = lc < ln_min ? ln_min : (lc > ln_max ? ln_max : lc);
            const float L = lookup_ln<R, float>(tab, T.n, lc, ln_min, inv_delta);
            d[v] = c2[v] < T.c2_event_min ? 0.0f : (float)rate_dt * expf(SPECIES == 1 ? L + lc : L) * (float)inv_g[v];
        }
    }
    if constexpr (SPECIES == 1) {
        // photons that cannot decay (R12) or lie outside the T table (Erber form): their value replaces
        // the clamped lookup's, one particle at a time -- the in-table photons of the warp pay nothing for them but the
        // branch (as rate_from_c2 decides, in its order)
        const double lo2 = T.chi_min * T.chi_min, hi2 = T.chi_max * T.chi_max;
#pragma unroll
        for (int v = 0; v < V; ++v) {
            if (!(g2[v] > 4.0) || !(c2[v] > 0.0)) d[v] = (R)0;
            else if (c2[v] < lo2 || c2[v] > hi2)
                d[v] = (c2[v] < T.c2_event_min || c2[v] < 1.7777e-4) ? (R)0 : erber_decrement<R>(c2[v], inv_g[v], rate_dt);
        }
    }
}

// ---- fused evolve kernel ------------------------------------------------------------
// V = particles per 128-bit load of R; U = independent vectors per thread per tile.  A warp owns U*32*V
// contiguous particles of the tile (every load instruction still covers 512 contiguous bytes).
// EMIT: also append a record (momentum, chi^2, index in chunk) of every particle that fired to the staging
// segment of its 128-particle chunk, in index order (warp ballot/popc; no CTA barrier), for event_kernel.
// Requires U*32*V == kChunk.
template <typename R, typename TR, int SPECIES, int U, bool EMIT, bool SCALED>
__global__ void __launch_bounds__(kEvolveThreads, U > 2 ? 1 : ((sizeof(R) == 4 && U == 1) ? 3 : 2))
evolve_kernel(const EvolveArgs<R, TR> a) {
    constexpr int V = 16 / sizeof(R);
    constexpr int TILE = kEvolveThreads * V * U;
    constexpr int WCH = U * 32 * V;  // particles per warp per tile
    static_assert(!EMIT || WCH == kChunk, "record staging works on 128-particle chunks");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned long long mbar;
    __shared__ unsigned int warp_counts[kEvolveThreads / 32];
    __shared__ double tau_new_s[(EMIT && SPECIES == 0) ? kEvolveThreads / 32 : 1][(EMIT && SPECIES == 0) ? kStageCap : 1];

    const R* tab = a.tab.L;
    if (a.table_in_smem) {
        const unsigned bytes = ((unsigned)(a.tab.n * sizeof(R)) + 15u) & ~15u;
        stage_table_tma(smem_raw, a.tab.L, bytes, &mbar);
        tab = reinterpret_cast<const R*>(smem_raw);
    }

    const unsigned long long pol_stream = l2_policy_evict_first();
    const unsigned long long pol_keep = l2_policy_evict_last();
    (void)pol_keep;
    unsigned int fired = 0;
    const long long ntiles = (a.n + TILE - 1) / TILE;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const long long base = tile * TILE;
        if (base + TILE <= a.n) {
            Vec<R, V> q[9][U];
            Vec<TR, V> t[U];
            // all loads of the tile first: 10*U independent 128-bit requests per thread in flight
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const long long i = base + (long long)warp * WCH + (u * 32 + lane) * V;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    q[c][u] = ld_stream<R, V>(a.p[c] + i, pol_stream);
                    q[3 + c][u] = ld_stream<R, V>(a.e[c] + i, pol_stream);
                    q[6 + c][u] = ld_stream<R, V>(a.b[c] + i, pol_stream);
                }
                t[u] = ld_stream_rw<TR, V>(a.tau + i, pol_stream);
            }
            unsigned int fired_bits = 0;
            double c2s[U * V];
            {
                // all U*V particles of the thread at once (decrement_vec interleaves their dependent chains)
                R in[9][U * V], d[U * V];
#pragma unroll
                for (int c = 0; c < 9; ++c)
#pragma unroll
                    for (int u = 0; u < U; ++u)
#pragma unroll
                        for (int v = 0; v < V; ++v) in[c][u * V + v] = q[c][u].v[v];
                decrement_vec<R, SPECIES, SCALED, U * V>(in, tab, a.tab, a.rate_dt, a.units, d, c2s);
#pragma unroll
                for (int u = 0; u < U; ++u) {
#pragma unroll
                    for (int v = 0; v < V; ++v) {
                        const TR tn = t[u].v[v] - (TR)d[u * V + v];
                        t[u].v[v] = tn;
                        fired += tn < (TR)0 ? 1u : 0u;
                        if (EMIT && tn < (TR)0) fired_bits |= 1u << (u * V + v);
                    }
                }
            }
            if constexpr (EMIT) {
                // rank inside the warp's chunk, in index order (u, lane, v): ballot / popc
                const unsigned int lt = (1u << lane) - 1u;
                unsigned int rank_u[U], total = 0;
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    unsigned int below = 0, all = 0;
#pragma unroll
                    for (int v = 0; v < V; ++v) {
                        const unsigned int bal = __ballot_sync(0xffffffffu, (fired_bits >> (u * V + v)) & 1u);
                        below += __popc(bal & lt);
                        all += __popc(bal);
                    }
                    rank_u[u] = total + below;
                    total += all;
                }
                const long long chunk = (base + (long long)warp * WCH) / kChunk;
                if (lane == 0) {
                    const bool part_done = SPECIES == 1 ? a.remove_photons != 0 : a.redraw_tau != 0;
                    a.stage_cnt[chunk] = (unsigned short)(total <= (unsigned)kStageCap
                                                              ? (total > 0 && part_done ? (total | kStageParentDone) : total)
                                                              : (total | kStageNoRecords));
                    if (total > 0) atomicAdd(a.tile_sum + chunk / kEventTileChunks, total);
                }
                if (total > 0 && total <= (unsigned)kStageCap) {  // (overflow: the event kernel re-scans the chunk)
                    // records are assembled in this warp's shared-memory buffer (scattered writes are cheap there)
                    // and leave as one coalesced stream of 128-bit stores
                    StageRecord<R>* wbuf = reinterpret_cast<StageRecord<R>*>(smem_raw + a.table_bytes) + warp * kStageCap;
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        unsigned int r = rank_u[u];
#pragma unroll
                        for (int v = 0; v < V; ++v) {
                            if ((fired_bits >> (u * V + v)) & 1u) {
                                StageRecord<R>& rec = wbuf[r];
                                rec.p[0] = q[0][u].v[v];
                                rec.p[1] = q[1][u].v[v];
                                rec.p[2] = q[2][u].v[v];
                                rec.c2 = c2s[u * V + v];
                                rec.idx = (unsigned)((u * 32 + lane) * V + v);
                                rec.tau_ev = (double)t[u].v[v];
                                ++r;
                            }
                        }
                    }
                    if (SPECIES == 0 && a.redraw_tau) {
                        // the new optical depths of the chunk's leptons in one pass: lane r serves record r (<= kStageCap < 32)
                        __syncwarp();
                        TR* tnew = reinterpret_cast<TR*>(tau_new_s[warp]);
                        if (lane < (int)total) {
                            const unsigned long long id =
                                a.id_base + (unsigned long long)(base + (long long)warp * WCH + (long long)wbuf[lane].idx);
                            const Words4 w = qed_words(a.seed, id, a.step, 1, 0);
                            tnew[lane] = draw_tau<TR>(w.w[2], w.w[3]);
                        }
                        __syncwarp();
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            unsigned int r = rank_u[u];
#pragma unroll
                            for (int v = 0; v < V; ++v)
                                if ((fired_bits >> (u * V + v)) & 1u) t[u].v[v] = tnew[r++];
                        }
                    }
                    if (SPECIES == 1 && a.remove_photons) {
                        // a photon that decays is removed whatever the split of its energy: p = 0, tau = +inf
                        // go out from here, with the stores of the evolve pass and while the momentum sectors are in L2 --
                        // the event pass has no scattered store left (it undoes this for events beyond the capacity)
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            if ((fired_bits >> (u * V)) & ((1u << V) - 1u)) {
                                const long long i = base + (long long)warp * WCH + (u * 32 + lane) * V;
#pragma unroll
                                for (int c = 0; c < 3; ++c) {
                                    Vec<R, V> z = q[c][u];
#pragma unroll
                                    for (int v = 0; v < V; ++v)
                                        if ((fired_bits >> (u * V + v)) & 1u) z.v[v] = (R)0;
                                    st_vec<R, V>(const_cast<R*>(a.p[c]) + i, z);
                                }
#pragma unroll
                                for (int v = 0; v < V; ++v)
                                    if ((fired_bits >> (u * V + v)) & 1u) t[u].v[v] = (TR)INFINITY;
                            }
                        }
                    }
                    __syncwarp();
                    const uint4* src = reinterpret_cast<const uint4*>(wbuf);
                    uint4* dst = reinterpret_cast<uint4*>(a.stage_rec + chunk * a.stage_stride);
                    const unsigned int nvec = total * StageRecord<R>::kVecs;
                    for (unsigned int k = lane; k < nvec; k += 32) st_policy(dst + k, src[k], pol_keep);
                    __syncwarp();
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const long long i = base + (long long)warp * WCH + (u * 32 + lane) * V;
                st_vec<TR, V>(a.tau + i, t[u]);
            }
        } else {  // ragged last tile: scalar, guarded (qed_step counts its chunks afterwards: count_chunks_kernel)
            for (long long i = base + threadIdx.x; i < a.n; i += kEvolveThreads) {
                const R d = decrement_one<R, SPECIES, SCALED>(a.p[0][i], a.p[1][i], a.p[2][i], a.e[0][i], a.e[1][i],
                                                      a.e[2][i], a.b[0][i], a.b[1][i], a.b[2][i], tab, a.tab,
                                                      a.rate_dt, a.units);
                const TR tn = a.tau[i] - (TR)d;
                a.tau[i] = tn;
                fired += tn < (TR)0 ? 1u : 0u;
            }
        }
    }

    if (a.d_n_events == nullptr) return;
    // CTA count -> partials[blockIdx]; the last CTA to arrive sums them in index order
    fired = __reduce_add_sync(0xffffffffu, fired);
    if ((threadIdx.x & 31) == 0) warp_counts[threadIdx.x >> 5] = fired;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int s = 0;
#pragma unroll
        for (int w = 0; w < kEvolveThreads / 32; ++w) s += warp_counts[w];
        a.partials[blockIdx.x] = s;
        __threadfence();
        const unsigned int arrived = atomicInc(a.ticket, gridDim.x - 1);  // wraps to 0 after the last CTA
        if (arrived == gridDim.x - 1) {
            __threadfence();
            unsigned long long total = 0;
            for (unsigned int k = 0; k < gridDim.x; ++k) total += ((volatile unsigned int*)a.partials)[k];
            *a.d_n_events = total;
        }
    }
}

// ---- standalone chi (PAPER.md:70 eq.2, :77 eq.3) ---------------------------------------
template <typename R, int SPECIES>
__global__ void __launch_bounds__(256) chi_kernel(const R* __restrict__ px, const R* __restrict__ py,
                                                  const R* __restrict__ pz, const R* __restrict__ ex,
                                                  const R* __restrict__ ey, const R* __restrict__ ez,
                                                  const R* __restrict__ bx, const R* __restrict__ by,
                                                  const R* __restrict__ bz, R* __restrict__ out, long long n,
                                                  const UnitScales us) {
    constexpr int V = 16 / sizeof(R);
    const long long nvec = n / V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    auto one = [&us](R pxr, R pyr, R pzr, R exr, R eyr, R ezr, R bxr, R byr, R bzr) -> R {
        const double x = pxr * us.p, y = pyr * us.p, z = pzr * us.p;
        const double p2 = fma(x, x, fma(y, y, z * z));
        const double g = sqrt(SPECIES == 0 ? 1.0 + p2 : p2);
        return (R)sqrt(chi_squared<SPECIES>(x, y, z, exr * us.e, eyr * us.e, ezr * us.e, bxr * us.b, byr * us.b,
                                            bzr * us.b, g, p2 > 1e-300 ? rcp_fast(p2) : 0.0));
    };
    const unsigned long long pol = l2_policy_evict_first();
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < nvec; j += stride) {
        const long long i = j * V;
        const Vec<R, V> a0 = ld_stream<R, V>(px + i, pol), a1 = ld_stream<R, V>(py + i, pol), a2 = ld_stream<R, V>(pz + i, pol),
                        a3 = ld_stream<R, V>(ex + i, pol), a4 = ld_stream<R, V>(ey + i, pol), a5 = ld_stream<R, V>(ez + i, pol),
                        a6 = ld_stream<R, V>(bx + i, pol), a7 = ld_stream<R, V>(by + i, pol), a8 = ld_stream<R, V>(bz + i, pol);
        Vec<R, V> o;
#pragma unroll
        for (int v = 0; v < V; ++v)
            o.v[v] = one(a0.v[v], a1.v[v], a2.v[v], a3.v[v], a4.v[v], a5.v[v], a6.v[v], a7.v[v], a8.v[v]);
        *reinterpret_cast<Vec<R, V>*>(out + i) = o;
    }
    // ragged tail
    for (long long i = nvec * V + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        out[i] = one(px[i], py[i], pz[i], ex[i], ey[i], ez[i], bx[i], by[i], bz[i]);
}

// ---- Schwinger pair-production rate per unit volume (eqs.19-22) ----------
// rate[i] = q_e^2 E_s^2/(4 pi^2 hbar^2 c) eps eta coth(pi eta/eps) exp(-pi/eps) in 1/(m^3 s), with
// F = (e^2 - b^2)/2, G = e.b, eps^2 = sqrt(F^2+G^2) + F, eta^2 = sqrt(F^2+G^2) - F.  The smaller of eps^2, eta^2 is
// taken as G^2 over the larger one (the literal difference cancels when abs(F) >> abs(G)).  Output is fp64 for
// either input type: the values span e^-600 .. 1e56.
constexpr double kSchwingerPrefactor =
    kElectronMass * kElectronMass * kElectronMass * kElectronMass * kLightSpeed * kLightSpeed * kLightSpeed *
    kLightSpeed * kLightSpeed /
    (4.0 * kPi * kPi * (kPlanck / (2.0 * kPi)) * (kPlanck / (2.0 * kPi)) * (kPlanck / (2.0 * kPi)) * (kPlanck / (2.0 * kPi)));

constexpr double kLnSchwingerPrefactor = 130.17295285072183;  // ln(kSchwingerPrefactor) (the parity test would show a slip)

__device__ __forceinline__ double schwinger_rate_one(double ex, double ey, double ez, double bx, double by, double bz) {
    const double e2 = fma(ex, ex, fma(ey, ey, ez * ez)), b2 = fma(bx, bx, fma(by, by, bz * bz));
    const double F = 0.5 * (e2 - b2), G = fma(ex, bx, fma(ey, by, ez * bz));
    const double s1 = fma(F, F, G * G);
    if (!(s1 > 1e-280)) return 0.0;                       // null field: eps = eta = 0
    const double big = s1 * rsqrt_fast(s1) + fabs(F);     // the larger of eps^2, eta^2
    const double small = G * G * rcp_fast(big);
    const double eps2 = F >= 0.0 ? big : small, eta2 = F >= 0.0 ? small : big;
    if (!(eps2 > 1e-280)) return 0.0;                     // exp(-pi/eps) = 0
    const double inv_eps = rsqrt_fast(eps2);
    const double eps = eps2 * inv_eps;
    const double eta = eta2 > 1e-280 ? eta2 * rsqrt_fast(eta2) : 0.0;
    const double x = kPi * eta * inv_eps;
    double eta_coth;                                      // eta coth(x); x coth x = 1 + x^2/3 - ... at x -> 0
    if (x > 1e-4) {
        const double q = exp_fast(-2.0 * x);
        eta_coth = eta * (1.0 + q) * rcp_fast(1.0 - q);
    } else {
        eta_coth = eps * (1.0 / kPi) * fma(x * x, 1.0 / 3.0, 1.0);
    }
    // the prefactor (~3e56) goes into the exponent: exp(-pi/eps) alone underflows long before the rate does
    return eps * eta_coth * exp_fast(kLnSchwingerPrefactor - kPi * inv_eps);
}

template <typename R>
__global__ void __launch_bounds__(256) schwinger_kernel(const R* __restrict__ ex, const R* __restrict__ ey,
                                                        const R* __restrict__ ez, const R* __restrict__ bx,
                                                        const R* __restrict__ by, const R* __restrict__ bz,
                                                        double* __restrict__ out, long long n, const UnitScales us) {
    constexpr int V = 16 / sizeof(R);
    const long long nvec = n / V;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const unsigned long long pol = l2_policy_evict_first();
    const double se = us.e, sb = us.b;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < nvec; j += stride) {
        const long long i = j * V;
        const Vec<R, V> a0 = ld_stream<R, V>(ex + i, pol), a1 = ld_stream<R, V>(ey + i, pol), a2 = ld_stream<R, V>(ez + i, pol),
                        a3 = ld_stream<R, V>(bx + i, pol), a4 = ld_stream<R, V>(by + i, pol), a5 = ld_stream<R, V>(bz + i, pol);
#pragma unroll
        for (int v = 0; v < V; v += 2) {
            double2 o;
            o.x = schwinger_rate_one(a0.v[v] * se, a1.v[v] * se, a2.v[v] * se, a3.v[v] * sb, a4.v[v] * sb, a5.v[v] * sb);
            o.y = schwinger_rate_one(a0.v[v + 1] * se, a1.v[v + 1] * se, a2.v[v + 1] * se, a3.v[v + 1] * sb, a4.v[v + 1] * sb,
                                     a5.v[v + 1] * sb);
            *reinterpret_cast<double2*>(out + i + v) = o;
        }
    }
    for (long long i = nvec * V + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        out[i] = schwinger_rate_one(ex[i] * se, ey[i] * se, ez[i] * se, bx[i] * sb, by[i] * sb, bz[i] * sb);
}

// ---- tau = -ln U, purpose 0, step 0 -------------------------------
template <typename TR>
__global__ void __launch_bounds__(256) init_tau_kernel(TR* __restrict__ tau, long long n, unsigned long long seed,
                                                       unsigned long long id_base, int species) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const Words4 w = qed_words(seed, id_base + (unsigned long long)i, 0ull, 0, species);
        tau[i] = draw_tau<TR>(w.w[0], w.w[1]);
    }
}

}  // namespace pxq
