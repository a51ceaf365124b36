// =====================================================================================
//  events.cuh -- event generation with deterministic stream compaction
//  (SURVEY.md 8(a) rows a5-a9): for every particle with tau < 0, inverse-CDF sampling of
//  the photon energy (eqs.28-30) or of the pair energy split
//  (eqs.24-26), creation of the secondaries in ascending parent index,
//  and the re-draw tau = -ln U.
//
//  One kernel, one pass over tau.  Per tile of 4096 particles: warp ballot/popc gives every
//  fired particle its rank inside its warp, a CTA-level scan of the 128 warp counts gives
//  the rank inside the tile, and a decoupled look-back over per-tile status words gives the
//  tile's offset in the output.  The fired particles of a tile are then gathered into a
//  dense list in shared memory so that full warps run the (branchy) binary search.
// =====================================================================================
#pragma once
#include "qed_device.cuh"
#include "evolve.cuh"

namespace pxq {

constexpr int kEventThreads = 256;
constexpr int kEventItems = 16;
constexpr int kEventTile = kEventThreads * kEventItems;  // 4096 particles
constexpr int kEventWarps = kEventThreads / 32;
constexpr int kEventChunks = kEventItems * kEventWarps;  // 128 (round, warp) chunks per tile

// look-back status word: [63:62] flag, [61:40] launch epoch, [39:0] count
constexpr unsigned long long kFlagAggregate = 1ull, kFlagInclusive = 2ull;
constexpr int kEpochBits = 22;
constexpr unsigned long long kValueMask = (1ull << 40) - 1;
__device__ __forceinline__ unsigned long long pack_status(unsigned long long flag, unsigned epoch,
                                                          unsigned long long value) {
    return (flag << 62) | ((unsigned long long)epoch << 40) | (value & kValueMask);
}

template <typename R, typename TR>
struct EventArgs {
    R* p[3];
    const R* e[3];
    const R* b[3];
    TR* tau;
    long long n;
    Table2D<R> cdf;
    unsigned long long seed, step, id_base;
    long long capacity;
    R* out_p[6];      // QS: photon px,py,pz (0..2).  BW: electron (0..2), positron (3..5)
    TR* out_tau[2];   // QS: photon tau.            BW: electron, positron tau
    long long* parent;
    unsigned long long* d_n_out;
    unsigned long long* status;        // one word per tile (ctx scratch)
    unsigned long long* tile_counter;  // monotonically increasing ticket counter (ctx scratch)
    unsigned long long tile_base;      // value of *tile_counter when this launch starts
    unsigned epoch;
    // staged_event_kernel only: records written by evolve_kernel<..., EMIT> (see evolve.cuh)
    const R* stage_rec;
    const unsigned char* stage_idx;
    const unsigned short* stage_cnt;
    long long stage_stride;
};

__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// ---- photon emission by one lepton ------------------------------
template <typename R, typename TR>
__device__ __forceinline__ void qs_event_core(const EventArgs<R, TR>& a, long long i, long long slot, double px,
                                              double py, double pz, double ex, double ey, double ez, double bx,
                                              double by, double bz) {
    const double p2 = fma(px, px, fma(py, py, pz * pz));
    const double g = sqrt(1.0 + p2);
    const double c2 = chi_squared<0>(px, py, pz, ex, ey, ez, bx, by, bz, g, p2);
    const unsigned long long id = a.id_base + (unsigned long long)i;
    const Words4 w = qed_words(a.seed, id, a.step, 1, 0);
    const Words4 wc = qed_words(a.seed, id, a.step, 2, 0);
    const double r = (double)uniform_open<R>(w.w[0], w.w[1]);
    const double xi = qs_sample_xi(a.cdf, 0.5 * log(c2), r);
    const double pn = sqrt(p2);
    const double inv_pn = pn > 0.0 ? 1.0 / pn : 0.0;
    const double nx = px * inv_pn, ny = py * inv_pn, nz = pz * inv_pn;
    const double km1 = p2 / (g + 1.0);          // gamma - 1 without cancellation
    const double gph = km1 * xi;                // gamma_gamma = (gamma-1) xi
    const double k2 = km1 * (1.0 - xi);         // emitter kinetic energy after the emission
    const double pn2 = sqrt(k2 * (k2 + 2.0));   // sqrt(gamma'^2 - 1)
    a.out_p[0][slot] = (R)(gph * nx);           // emitted along p
    a.out_p[1][slot] = (R)(gph * ny);
    a.out_p[2][slot] = (R)(gph * nz);
    a.out_tau[0][slot] = draw_tau<TR>(wc.w[0], wc.w[1]);
    if (a.parent) a.parent[slot] = i;
    a.p[0][i] = (R)(pn2 * nx);
    a.p[1][i] = (R)(pn2 * ny);
    a.p[2][i] = (R)(pn2 * nz);
    a.tau[i] = draw_tau<TR>(w.w[2], w.w[3]);
}
template <typename R, typename TR>
__device__ __forceinline__ void qs_event(const EventArgs<R, TR>& a, long long i, long long slot) {
    qs_event_core<R, TR>(a, i, slot, a.p[0][i], a.p[1][i], a.p[2][i], a.e[0][i], a.e[1][i], a.e[2][i], a.b[0][i],
                         a.b[1][i], a.b[2][i]);
}

// ---- pair production by one photon -----------------------------
template <typename R, typename TR>
__device__ __forceinline__ void bw_event_core(const EventArgs<R, TR>& a, long long i, long long slot, double px,
                                              double py, double pz, double ex, double ey, double ez, double bx,
                                              double by, double bz) {
    const double p2 = fma(px, px, fma(py, py, pz * pz));
    const double g = sqrt(p2);                  // gamma_gamma = |p|
    const double c2 = chi_squared<1>(px, py, pz, ex, ey, ez, bx, by, bz, g, p2);
    const unsigned long long id = a.id_base + (unsigned long long)i;
    const Words4 w = qed_words(a.seed, id, a.step, 1, 1);
    const Words4 wc = qed_words(a.seed, id, a.step, 2, 1);
    const double r = (double)uniform_open<R>(w.w[0], w.w[1]);
    const bool electron_side = r <= 0.5;        // PAPER.md:212 "If r <= 0.5"
    const double rp = electron_side ? r : 1.0 - r;
    const double xi = bw_sample_xi(a.cdf, 0.5 * log(c2), rp);
    const double xe = electron_side ? xi : 1.0 - xi;   // chi_-/chi_gamma
    const double xp = electron_side ? 1.0 - xi : xi;   // chi_+/chi_gamma (eq.6)
    const double ke = (g - 2.0) * xe, kp = (g - 2.0) * xp;  // K = (gamma_gamma-2) chi_pm/chi_gamma
    const double pe = sqrt(ke * (ke + 2.0)), pp = sqrt(kp * (kp + 2.0));
    const double inv_g = g > 0.0 ? 1.0 / g : 0.0;
    const double nx = px * inv_g, ny = py * inv_g, nz = pz * inv_g;
    a.out_p[0][slot] = (R)(pe * nx);
    a.out_p[1][slot] = (R)(pe * ny);
    a.out_p[2][slot] = (R)(pe * nz);
    a.out_p[3][slot] = (R)(pp * nx);
    a.out_p[4][slot] = (R)(pp * ny);
    a.out_p[5][slot] = (R)(pp * nz);
    a.out_tau[0][slot] = draw_tau<TR>(wc.w[0], wc.w[1]);
    a.out_tau[1][slot] = draw_tau<TR>(wc.w[2], wc.w[3]);
    if (a.parent) a.parent[slot] = i;
    a.p[0][i] = (R)0;                           // photon removed: p = 0, tau = +inf
    a.p[1][i] = (R)0;
    a.p[2][i] = (R)0;
    a.tau[i] = (TR)INFINITY;
}
template <typename R, typename TR>
__device__ __forceinline__ void bw_event(const EventArgs<R, TR>& a, long long i, long long slot) {
    bw_event_core<R, TR>(a, i, slot, a.p[0][i], a.p[1][i], a.p[2][i], a.e[0][i], a.e[1][i], a.e[2][i], a.b[0][i],
                         a.b[1][i], a.b[2][i]);
}

// ---- decoupled look-back over the per-tile status words (one full warp) --------------------
// Publishes `total` as this tile's aggregate, sums the counts of all earlier tiles (waiting only for tiles that
// were handed out before this one, hence already running), publishes the inclusive prefix and returns the
// exclusive one in every lane.
__device__ __forceinline__ unsigned long long tile_exclusive_prefix(unsigned long long* status, long long tile,
                                                                    unsigned epoch, unsigned long long total, int lane) {
    unsigned long long excl = 0;
    if (tile == 0) {
        if (lane == 0) st_relaxed(status, pack_status(kFlagInclusive, epoch, total));
        return 0;
    }
    if (lane == 0) st_relaxed(status + tile, pack_status(kFlagAggregate, epoch, total));
    long long look = tile - 1;  // lane l inspects tile look - l
    while (true) {
        const long long idx = look - lane;
        unsigned long long word = 0;
        bool ready;
        do {  // wait until every inspected predecessor has published for this launch
            ready = true;
            if (idx >= 0) {
                word = ld_relaxed(status + idx);
                ready = (word >> 62) != 0 && (unsigned)((word >> 40) & ((1u << kEpochBits) - 1)) == epoch;
            }
        } while (!__all_sync(0xffffffffu, ready));
        const bool inclusive = idx >= 0 && (word >> 62) == kFlagInclusive;
        const unsigned int inc_mask = __ballot_sync(0xffffffffu, inclusive);
        const int stop = inc_mask ? __ffs(inc_mask) - 1 : 31;  // nearest inclusive prefix
        unsigned long long v = (idx >= 0 && lane <= stop) ? (word & kValueMask) : 0ull;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        excl += v;
        if (inc_mask || look - 32 < 0) break;
        look -= 32;
    }
    if (lane == 0) st_relaxed(status + tile, pack_status(kFlagInclusive, epoch, excl + total));
    return excl;
}

// ---- the event kernel ------------------------------------------------------------------
// KIND 0: photon emission by leptons; KIND 1: pair production by photons.
template <typename R, typename TR, int KIND>
__global__ void __launch_bounds__(kEventThreads) event_kernel(const EventArgs<R, TR> a) {
    __shared__ unsigned int chunk_off[kEventChunks];   // counts, then exclusive offsets, in (round, warp) order
    __shared__ unsigned short list[kEventTile];        // tile-local indices of the fired particles, ascending
    __shared__ long long s_tile;
    __shared__ unsigned long long s_excl;               // number of fired particles in all earlier tiles
    __shared__ unsigned int s_total;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // tiles are handed out in launch order, so every tile's predecessors are already running
    if (tid == 0) s_tile = (long long)(atomicAdd(a.tile_counter, 1ull) - a.tile_base);
    __syncthreads();
    const long long tile = s_tile;
    const long long base = tile * kEventTile;

    // 1. flags: tau < 0 (R1).  All loads first.
    TR t[kEventItems];
#pragma unroll
    for (int j = 0; j < kEventItems; ++j) {
        const long long i = base + j * kEventThreads + tid;
        t[j] = i < a.n ? a.tau[i] : (TR)1;
    }
    unsigned int my_flags = 0;
    unsigned int my_rank[kEventItems / 4];  // 8-bit lane ranks (< 32), packed
#pragma unroll
    for (int j = 0; j < kEventItems / 4; ++j) my_rank[j] = 0;
#pragma unroll
    for (int j = 0; j < kEventItems; ++j) {
        const bool f = t[j] < (TR)0;
        const unsigned int bal = __ballot_sync(0xffffffffu, f);
        if (f) my_flags |= 1u << j;
        my_rank[j >> 2] |= (unsigned)__popc(bal & ((1u << lane) - 1u)) << (8 * (j & 3));
        if (lane == 0) chunk_off[j * kEventWarps + warp] = __popc(bal);
    }
    __syncthreads();

    // 2. CTA scan of the 128 chunk counts (warp 0: 4 per lane + shuffle scan)
    if (warp == 0) {
        unsigned int c[4], s = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) { c[k] = chunk_off[4 * lane + k]; s += c[k]; }
        unsigned int incl = s;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned int o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        unsigned int run = incl - s;
#pragma unroll
        for (int k = 0; k < 4; ++k) { chunk_off[4 * lane + k] = run; run += c[k]; }
        const unsigned int total = __shfl_sync(0xffffffffu, incl, 31);

        // 3. decoupled look-back: publish this tile's count, then sum the predecessors'
        const unsigned long long excl = tile_exclusive_prefix(a.status, tile, a.epoch, total, lane);
        if (lane == 0) {
            s_excl = excl;
            s_total = total;
            if (base + kEventTile >= a.n) *a.d_n_out = excl + total;  // last tile: total fired
        }
    }
    __syncthreads();

    // 4. gather the fired particles of the tile into a dense, index-ordered list
#pragma unroll
    for (int j = 0; j < kEventItems; ++j) {
        if (my_flags & (1u << j)) {
            const unsigned int rank = (my_rank[j >> 2] >> (8 * (j & 3))) & 0xffu;
            list[chunk_off[j * kEventWarps + warp] + rank] = (unsigned short)(j * kEventThreads + tid);
        }
    }
    __syncthreads();

    // 5. events, densely packed over the threads; slot = number of fired particles before this one
    const unsigned int total = s_total;
    const unsigned long long excl = s_excl;
    for (unsigned int q = tid; q < total; q += kEventThreads) {
        const long long slot = (long long)(excl + q);
        if (slot >= a.capacity) break;  // capacity rule: later parents are left untouched
        const long long i = base + list[q];
        if (KIND == 0) qs_event<R, TR>(a, i, slot); else bw_event<R, TR>(a, i, slot);
    }
}

// ---- events from staged records -----------------------------------------------------------
// Second half of picsarqed_qed_step.  evolve_kernel<..., EMIT> has already written, for every 128-particle
// chunk, the number of particles that fired and their nine reals (in index order).  One CTA owns a tile of
// 4096 particles = 32 chunks: it sums the 32 counts, gets the tile's output offset from the decoupled
// look-back and runs the events densely over its threads, reading coalesced records instead of scanning
// tau and gathering scattered particles.  Chunks whose segment overflowed (more than kStageCap events) or
// that belong to the ragged tail are re-scanned from tau, exactly like event_kernel does.
constexpr int kTileChunks = kEventTile / kChunk;  // 32

template <typename R, typename TR, int KIND>
__global__ void __launch_bounds__(kEventThreads) staged_event_kernel(const EventArgs<R, TR> a) {
    __shared__ unsigned int cnt[kTileChunks];
    __shared__ unsigned int off[kTileChunks + 1];
    __shared__ unsigned char rescan[kTileChunks];
    __shared__ unsigned char list[kTileChunks][kChunk];  // re-scanned chunks: local indices of the fired particles
    __shared__ long long s_tile;
    __shared__ unsigned long long s_excl;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = (long long)(atomicAdd(a.tile_counter, 1ull) - a.tile_base);
    __syncthreads();
    const long long tile = s_tile;
    const long long first_chunk = tile * kTileChunks;

    // 1. per-chunk counts (4 chunks per warp); overflowed / tail chunks are re-scanned with ballot/popc
#pragma unroll 1
    for (int k = 0; k < kTileChunks / kEventWarps; ++k) {
        const int j = warp * (kTileChunks / kEventWarps) + k;
        const long long cbase = (first_chunk + j) * kChunk;
        unsigned int c = cbase < a.n ? a.stage_cnt[first_chunk + j] : 0u;
        const bool re = c > (unsigned)kStageCap;
        if (re) {
            c = 0;
#pragma unroll
            for (int r4 = 0; r4 < kChunk / 32; ++r4) {
                const long long i = cbase + r4 * 32 + lane;
                const bool f = i < a.n && a.tau[i] < (TR)0;
                const unsigned int bal = __ballot_sync(0xffffffffu, f);
                if (f) list[j][c + __popc(bal & ((1u << lane) - 1u))] = (unsigned char)(r4 * 32 + lane);
                c += __popc(bal);
            }
        }
        if (lane == 0) { cnt[j] = c; rescan[j] = re ? 1 : 0; }
    }
    __syncthreads();

    // 2. offsets of the chunks inside the tile, offset of the tile in the output (decoupled look-back)
    if (warp == 0) {
        const unsigned int c = cnt[lane];
        unsigned int incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned int o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        off[lane] = incl - c;
        const unsigned int total = __shfl_sync(0xffffffffu, incl, 31);
        if (lane == 31) off[kTileChunks] = total;
        const unsigned long long excl = tile_exclusive_prefix(a.status, tile, a.epoch, total, lane);
        if (lane == 0) {
            s_excl = excl;
            if ((tile + 1) * (long long)kEventTile >= a.n) *a.d_n_out = excl + total;  // last tile: total fired
        }
    }
    __syncthreads();

    // 3. events, densely over the threads
    const unsigned int total = off[kTileChunks];
    const unsigned long long excl = s_excl;
    for (unsigned int e = tid; e < total; e += kEventThreads) {
        const long long slot = (long long)(excl + e);
        if (slot >= a.capacity) break;  // capacity rule (R16)
        int j = 0;                      // largest j with off[j] <= e
#pragma unroll
        for (int step = kTileChunks / 2; step > 0; step >>= 1)
            if (off[j + step] <= e) j += step;
        const unsigned int r = e - off[j];
        const long long cbase = (first_chunk + j) * kChunk;
        double px, py, pz, ex, ey, ez, bx, by, bz;
        long long i;
        if (rescan[j]) {
            i = cbase + list[j][r];
            px = a.p[0][i]; py = a.p[1][i]; pz = a.p[2][i];
            ex = a.e[0][i]; ey = a.e[1][i]; ez = a.e[2][i];
            bx = a.b[0][i]; by = a.b[1][i]; bz = a.b[2][i];
        } else {
            const long long pos = (first_chunk + j) * kStageCap + r;
            i = cbase + a.stage_idx[pos];
            const R* rec = a.stage_rec + pos;
            px = rec[0]; py = rec[a.stage_stride]; pz = rec[2 * a.stage_stride];
            ex = rec[3 * a.stage_stride]; ey = rec[4 * a.stage_stride]; ez = rec[5 * a.stage_stride];
            bx = rec[6 * a.stage_stride]; by = rec[7 * a.stage_stride]; bz = rec[8 * a.stage_stride];
        }
        if (KIND == 0) qs_event_core<R, TR>(a, i, slot, px, py, pz, ex, ey, ez, bx, by, bz);
        else bw_event_core<R, TR>(a, i, slot, px, py, pz, ex, ey, ez, bx, by, bz);
    }
}

}  // namespace pxq
