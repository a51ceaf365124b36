// =====================================================================================
//  events.cuh -- event generation with deterministic stream compaction
//  (SURVEY.md 8(a) rows a5-a9): for every particle with tau < 0, inverse-CDF sampling of
//  the photon energy (eqs.28-30) or of the pair energy split
//  (eqs.24-26), creation of the secondaries in ascending parent index,
//  and the re-draw tau = -ln U.
//
//  Compaction in three levels, all deterministic:
//   1. warp ballot/popc ranks the fired particles of a 128-particle chunk and counts them
//      (inside the evolve pass for picsarqed_qed_step, count_chunks_kernel for generate_*);
//   2. tile_scan_kernel: one CTA sums the chunk counts per tile and scans the tile sums
//      (block-level scan) into exclusive output offsets and the total;
//   3. event_kernel: a tile of consecutive chunks per CTA; event e of the tile is handled by
//      thread e, its output slot is tile_offset + e.  Tiles are independent: no
//      ticket, no look-back, no barrier on the common path.
//  (A single-pass decoupled look-back was tried first: with ~10^3 tiles in flight every tile
//  walks ~30 status windows before it meets an inclusive prefix, which serialised the kernel
//  at ~0.3 ms per 16 Mi particles whatever its shape (round-1 capture).)
// =====================================================================================
#pragma once
#include "qed_device.cuh"
#include "evolve.cuh"

namespace pxq {

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
    // per 128-particle chunk (context scratch, see evolve.cuh):
    const unsigned char* stage_rec;           // staged records (unused for chunks flagged kStageNoRecords), or, for
                                              // chunks flagged kStageDone, staged StepResult records (fused step)
    long long stage_stride;                   // bytes from one chunk's segment to the next
    const unsigned short* stage_cnt;          // count | flags
    const unsigned long long* tile_offset;    // [n_tiles] number of events before the tile
    // a call that handles the slab [parent_base, parent_base + n) of a longer array (step_host): its events
    // follow the *slot_base events of the slabs before it (device word, NULL = 0), parents are numbered globally
    const unsigned long long* slot_base;
    long long parent_base;
    UnitScales units;   // the caller's unit system: momenta and fields are scaled where they are loaded, momenta back
                        // where they are stored; the event arithmetic itself is in the library's units
};

template <typename R, typename TR>
struct EventOut {
    R sec[6];     // QS: photon momentum (0..2).  BW: electron (0..2) and positron (3..5) momenta
    TR sec_tau[2];
    R parent_p[3];
    TR parent_tau;
};

// ---- photon emission by one lepton ------------------------------
template <typename R, typename TR>
__device__ __forceinline__ EventOut<R, TR> qs_event_compute(const EventArgs<R, TR>& a, long long i, double px, double py,
                                                            double pz, double c2) {
    // (lean fp64 routines of qed_device.cuh: every argument here is a positive normal number or handled apart)
    const double p2 = fma(px, px, fma(py, py, pz * pz));
    const double g = (1.0 + p2) * rsqrt_fast(1.0 + p2);
    const unsigned long long id = a.id_base + (unsigned long long)i;
    const Words4 w = qed_words(a.seed, id, a.step, 1, 0);
    const Words4 wc = qed_words(a.seed, id, a.step, 2, 0);
    const double r = (double)uniform_open<R>(w.w[0], w.w[1]);
    // the logarithms of the event at once (ln r, ln chi^2 and, for an fp64 optical depth, the two re-draws): four
    // independent chains the V-at-once routine interleaves
    double lg[4];
    if constexpr (sizeof(TR) == 8) {
        const double la[4] = {r, c2, uniform_open<double>(w.w[2], w.w[3]), uniform_open<double>(wc.w[0], wc.w[1])};
        log_pos_v<4>(la, lg);
    } else {
        const double la[2] = {r, c2};
        double l2[2];
        log_pos_v<2>(la, l2);
        lg[0] = l2[0]; lg[1] = l2[1]; lg[2] = lg[3] = 0.0;
    }
    const double xi = qs_sample_xi_ln(a.cdf, 0.5 * lg[1], lg[0], r);
    const double inv_pn = p2 > 1e-300 ? rsqrt_fast(p2) : 0.0;
    const double nx = px * inv_pn, ny = py * inv_pn, nz = pz * inv_pn;
    const double km1 = p2 * rcp_fast(g + 1.0);  // gamma - 1 without cancellation
    const double gph = km1 * xi;                // gamma_gamma = (gamma-1) xi
    const double k2 = km1 * (1.0 - xi);         // emitter kinetic energy after the emission
    const double q2 = k2 * (k2 + 2.0);
    const double pn2 = q2 > 1e-300 ? q2 * rsqrt_fast(q2) : 0.0;   // sqrt(gamma'^2 - 1)
    EventOut<R, TR> o;
    const double ip = a.units.inv_p;
    o.sec[0] = (R)(gph * nx * ip);              // emitted along p
    o.sec[1] = (R)(gph * ny * ip);
    o.sec[2] = (R)(gph * nz * ip);
    o.sec[3] = o.sec[4] = o.sec[5] = (R)0;
    if constexpr (sizeof(TR) == 8) o.sec_tau[0] = -lg[3]; else o.sec_tau[0] = draw_tau<TR>(wc.w[0], wc.w[1]);
    o.sec_tau[1] = (TR)0;
    o.parent_p[0] = (R)(pn2 * nx * ip);
    o.parent_p[1] = (R)(pn2 * ny * ip);
    o.parent_p[2] = (R)(pn2 * nz * ip);
    if constexpr (sizeof(TR) == 8) o.parent_tau = -lg[2]; else o.parent_tau = draw_tau<TR>(w.w[2], w.w[3]);
    return o;
}

// ---- pair production by one photon -----------------------------
template <typename R, typename TR>
__device__ __forceinline__ EventOut<R, TR> bw_event_compute(const EventArgs<R, TR>& a, long long i, double px, double py,
                                                            double pz, double c2) {
    const double p2 = fma(px, px, fma(py, py, pz * pz));
    const double inv_g = p2 > 1e-300 ? rsqrt_fast(p2) : 0.0;
    const double g = p2 * inv_g;                // gamma_gamma = |p|
    const unsigned long long id = a.id_base + (unsigned long long)i;
    const Words4 w = qed_words(a.seed, id, a.step, 1, 1);
    const Words4 wc = qed_words(a.seed, id, a.step, 2, 1);
    const double r = (double)uniform_open<R>(w.w[0], w.w[1]);
    const bool electron_side = r <= 0.5;        // PAPER.md:212 "If r <= 0.5"
    const double rp = electron_side ? r : 1.0 - r;
    double lg[3];
    if constexpr (sizeof(TR) == 8) {
        const double la[3] = {c2, uniform_open<double>(wc.w[0], wc.w[1]), uniform_open<double>(wc.w[2], wc.w[3])};
        log_pos_v<3>(la, lg);
    } else {
        lg[0] = log_pos(c2); lg[1] = lg[2] = 0.0;
    }
    const double xi = bw_sample_xi(a.cdf, 0.5 * lg[0], rp);
    const double xe = electron_side ? xi : 1.0 - xi;   // chi_-/chi_gamma
    const double xp = electron_side ? 1.0 - xi : xi;   // chi_+/chi_gamma (eq.6)
    const double ke = (g - 2.0) * xe, kp = (g - 2.0) * xp;  // K = (gamma_gamma-2) chi_pm/chi_gamma
    const double qe = ke * (ke + 2.0), qp = kp * (kp + 2.0);
    const double pe = qe > 1e-300 ? qe * rsqrt_fast(qe) : 0.0, pp = qp > 1e-300 ? qp * rsqrt_fast(qp) : 0.0;
    const double nx = px * inv_g, ny = py * inv_g, nz = pz * inv_g;
    EventOut<R, TR> o;
    const double ip = a.units.inv_p;
    o.sec[0] = (R)(pe * nx * ip);
    o.sec[1] = (R)(pe * ny * ip);
    o.sec[2] = (R)(pe * nz * ip);
    o.sec[3] = (R)(pp * nx * ip);
    o.sec[4] = (R)(pp * ny * ip);
    o.sec[5] = (R)(pp * nz * ip);
    if constexpr (sizeof(TR) == 8) { o.sec_tau[0] = -lg[1]; o.sec_tau[1] = -lg[2]; }
    else { o.sec_tau[0] = draw_tau<TR>(wc.w[0], wc.w[1]); o.sec_tau[1] = draw_tau<TR>(wc.w[2], wc.w[3]); }
    o.parent_p[0] = o.parent_p[1] = o.parent_p[2] = (R)0;   // photon removed: p = 0, tau = +inf
    o.parent_tau = (TR)INFINITY;
    return o;
}

// chi^2 of a parent gathered from the particle arrays (chunks without staged records)
template <int KIND>
__device__ __forceinline__ double event_c2(double px, double py, double pz, double ex, double ey, double ez, double bx,
                                           double by, double bz) {
    double inv_g, g2;
    return chi_squared_of<KIND>(px, py, pz, ex, ey, ez, bx, by, bz, &inv_g, &g2);
}

template <typename R, typename TR, int KIND>
__device__ __forceinline__ void event_commit(const EventArgs<R, TR>& a, long long i, long long slot,
                                             const EventOut<R, TR>& o, bool parent_done = false) {
#pragma unroll
    for (int c = 0; c < (KIND == 0 ? 3 : 6); ++c) a.out_p[c][slot] = o.sec[c];
    a.out_tau[0][slot] = o.sec_tau[0];
    if (KIND == 1) a.out_tau[1][slot] = o.sec_tau[1];
    if (a.parent) a.parent[slot] = a.parent_base + i;
    if (parent_done && KIND == 1) return;   // (a photon the evolve pass removed itself)
#pragma unroll
    for (int c = 0; c < 3; ++c) a.p[c][i] = o.parent_p[c];
    if (!parent_done) a.tau[i] = o.parent_tau;   // (parent_done, lepton: the evolve pass stored the new optical depth itself)
}

// ---- level 1 for generate_*: count the fired particles of every chunk --------------------------
// one warp per chunk: tau < 0 (R1) -> ballot/popc.  No records are staged on this path.
template <typename TR>
__global__ void __launch_bounds__(256) count_chunks_kernel(const TR* __restrict__ tau, long long n, long long first_chunk,
                                                           long long n_chunks, unsigned short* __restrict__ cnt,
                                                           unsigned int* __restrict__ tile_sum, int chunks_per_tile) {
    const int lane = threadIdx.x & 31;
    const long long warps = (long long)gridDim.x * (blockDim.x / 32);
    for (long long ch = first_chunk + (long long)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5); ch < n_chunks; ch += warps) {
        unsigned int k = 0;
#pragma unroll
        for (int r4 = 0; r4 < kChunk / 32; ++r4) {
            const long long i = ch * kChunk + r4 * 32 + lane;
            const bool f = i < n && tau[i] < (TR)0;
            k += __popc(__ballot_sync(0xffffffffu, f));
        }
        if (lane == 0) {
            cnt[ch] = (unsigned short)(k | kStageNoRecords);
            if (k > 0) atomicAdd(tile_sum + ch / chunks_per_tile, k);   // (see EvolveArgs::tile_sum)
        }
    }
}

// ---- level 2: output offsets of the tiles (block-level scan) -------------------------------------
// tile_scan_kernel: one CTA sums the chunk counts of every tile (128-bit loads of eight 16-bit counts when a tile
// is a multiple of 8 chunks) and scans the tile sums, 4096 tiles per round (four consecutive tiles per thread),
// carrying the running total; tile_offset[t] = number of events before tile t, *d_total = *d_base (0 when
// d_base is NULL) + their number.  d_base chains the slabs of step_host: the events of a slab follow those of
// the slabs before it in the secondary buffers.  d_entries (not NULL: the append of cascade.cuh) = device count of
// the entries that exist: only the chunks that hold them are read.  tile_sum (not NULL: the QED step) holds the tile
// sums already, accumulated by the kernels that counted the chunks; they are read instead of the 16-bit counts
// (one word per tile: the scan of 16 Mi particles reads 22 KB instead of 262 KB through its single CTA) and
// reset to zero for the next call.
constexpr int kScanThreads = 1024;
constexpr int kScanItems = 4;

__global__ void __launch_bounds__(kScanThreads) tile_scan_kernel(const unsigned short* __restrict__ cnt, long long n_chunks,
                                                                 int chunks_per_tile, long long n_tiles,
                                                                 unsigned long long* __restrict__ tile_offset,
                                                                 const unsigned long long* d_base,
                                                                 unsigned long long* d_total,
                                                                 const unsigned long long* d_entries,
                                                                 unsigned int* __restrict__ tile_sum) {
    __shared__ unsigned long long warp_sum[2][kScanThreads / 32];
    asm volatile("griddepcontrol.launch_dependents;");   // (the event kernel may take its place on the SMs; it waits for this grid's end)
    if (d_entries) {
        const unsigned long long live = (*d_entries + kChunk - 1) / kChunk;
        if (live < (unsigned long long)n_chunks) n_chunks = (long long)live;
        n_tiles = (n_chunks + chunks_per_tile - 1) / chunks_per_tile;
    }
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long carry = 0;  // (the same value in every thread)
    int round = 0;
    // the tile sums of the next round are requested before this round is scanned: a round costs its shuffles and its
    // barrier, not a trip to L2 (256 Mi particles are 16 rounds)
    uint4 q_next = make_uint4(0u, 0u, 0u, 0u);
    if (tile_sum != nullptr && (long long)tid * kScanItems + kScanItems <= n_tiles)
        q_next = *reinterpret_cast<const uint4*>(tile_sum + (long long)tid * kScanItems);
    for (long long base = 0; base < n_tiles; base += kScanThreads * kScanItems, ++round) {
        const long long t0 = base + (long long)tid * kScanItems;
        unsigned int v[kScanItems];
        if (tile_sum != nullptr) {
            if (t0 + kScanItems <= n_tiles) {   // t0 is a multiple of 4: 16-byte aligned
                const uint4 q = q_next;
                const long long t1 = t0 + (long long)kScanThreads * kScanItems;
                if (t1 + kScanItems <= n_tiles) q_next = *reinterpret_cast<const uint4*>(tile_sum + t1);
                v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
                *reinterpret_cast<uint4*>(tile_sum + t0) = make_uint4(0u, 0u, 0u, 0u);
            } else {
#pragma unroll
                for (int k = 0; k < kScanItems; ++k) {
                    v[k] = t0 + k < n_tiles ? tile_sum[t0 + k] : 0u;
                    if (t0 + k < n_tiles) tile_sum[t0 + k] = 0u;
                }
            }
        } else
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            const long long c0 = (t0 + k) * chunks_per_tile;
            unsigned int sum = 0;
            if (t0 + k < n_tiles) {
                if ((chunks_per_tile & 7) == 0 && c0 + chunks_per_tile <= n_chunks) {
                    for (int c = 0; c < chunks_per_tile; c += 8) {  // 8 counts per 128-bit load, two per word
                        const uint4 q = *reinterpret_cast<const uint4*>(cnt + c0 + c);
                        const unsigned int w4[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
                        for (int j = 0; j < 4; ++j) sum += (w4[j] & kStageCountMask) + ((w4[j] >> 16) & kStageCountMask);
                    }
                } else {
                    for (long long c = c0; c < min(c0 + (long long)chunks_per_tile, n_chunks); ++c) sum += cnt[c] & kStageCountMask;
                }
            }
            v[k] = sum;
        }
        const unsigned long long s = (unsigned long long)v[0] + v[1] + v[2] + v[3];
        unsigned long long incl = s;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        if (lane == 31) warp_sum[round & 1][warp] = incl;
        __syncthreads();  // (double-buffered: one barrier per round)
        unsigned long long before = carry, all = 0;
#pragma unroll 8
        for (int w = 0; w < kScanThreads / 32; ++w) {
            const unsigned long long ws = warp_sum[round & 1][w];
            if (w < warp) before += ws;
            all += ws;
        }
        unsigned long long run = before + incl - s;
#pragma unroll
        for (int k = 0; k < kScanItems; ++k) {
            if (t0 + k < n_tiles) tile_offset[t0 + k] = run;
            run += v[k];
        }
        carry += all;
    }
    if (tid == 0) *d_total = (d_base ? *d_base : 0ull) + carry;
}

// ---- level 3: the events ---------------------------------------------------------------------
// THREADS threads own a tile of CHUNKS consecutive chunks (CHUNKS <= 32).  Lane j of every warp reads the
// count of chunk j (coalesced) and a warp scan gives the tile's layout, in registers, in every warp.  Event e of
// the tile (e = 0 .. total-1, normally one per thread) belongs to the chunk j with off_j <= e < off_{j+1};
// its data come from the staged record r = e - off_j of that chunk, or, when the chunk has no records
// (generate_* path, segment overflow, ragged tail), from a ballot/popc re-scan of the chunk's tau.
template <typename R, typename TR, int KIND, int THREADS, int CHUNKS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) event_kernel(const EventArgs<R, TR> a) {
    constexpr int WARPS = THREADS / 32;
    __shared__ unsigned char list[CHUNKS][kChunk];  // re-scanned chunks: local indices of the fired particles

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long n_chunks = (a.n + kChunk - 1) / kChunk;
    const long long n_tiles = (n_chunks + CHUNKS - 1) / CHUNKS;
    // launched as a programmatic dependent of tile_scan_kernel: everything before this line overlaps the scan; the tile
    // offsets (and everything the kernels before it wrote) are visible after it.  A no-op in an ordinary launch.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // Persistent CTAs stride over the tiles.  The warps of a CTA walk the same tiles in the same order but do
    // not wait for one another (no barrier on the common path): a warp whose slice of a tile holds no event is
    // already loading the next tile.  The loads of the next tile are issued before the current one is processed.
    auto load_flags = [&](long long tile) -> unsigned short {
        const long long ch = tile * CHUNKS + lane;
        return (tile < n_tiles && lane < CHUNKS && ch < n_chunks) ? a.stage_cnt[ch] : (unsigned short)0;
    };
    const unsigned long long slot_base = a.slot_base ? *a.slot_base : 0ull;
    // (the tiles are walked from the last one down: the particles the evolve pass streamed last are the ones whose
    // sectors may still be in L2 when their parents are rewritten)
#define PXQ_TILE_OF(it) (n_tiles - 1 - (it))
    long long it = blockIdx.x;
    unsigned short flags_next = it < n_tiles ? load_flags(PXQ_TILE_OF(it)) : (unsigned short)0;
    unsigned long long excl_next = it < n_tiles ? a.tile_offset[PXQ_TILE_OF(it)] : 0ull;
    for (; it < n_tiles; it += gridDim.x) {
    const long long tile = PXQ_TILE_OF(it);
    const long long first_chunk = tile * CHUNKS;
    const unsigned short flags = flags_next;
    const unsigned long long excl = excl_next;                            // output slot of the tile's first event
    const long long it_next = it + gridDim.x;
    flags_next = it_next < n_tiles ? load_flags(PXQ_TILE_OF(it_next)) : (unsigned short)0;
    excl_next = it_next < n_tiles ? a.tile_offset[PXQ_TILE_OF(it_next)] : 0ull;
    const unsigned int cnt = flags & kStageCountMask;
    unsigned int incl = cnt;                                             // offsets of the chunks inside the tile
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned int o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    const unsigned int off_lane = incl - cnt;
    const unsigned int total = __shfl_sync(0xffffffffu, incl, 31);
    if (total == 0) continue;
    unsigned int rescan_mask = 0, done_mask = 0, pdone_mask = 0;
    if (__any_sync(0xffffffffu, cnt > (unsigned)kStageCap || (flags & ~kStageCountMask) != 0)) {   // (rarely: most tiles are plain)
        rescan_mask = __ballot_sync(0xffffffffu, cnt > 0 && (cnt > (unsigned)kStageCap || (flags & kStageNoRecords) != 0));
        done_mask = __ballot_sync(0xffffffffu, cnt > 0 && (flags & kStageDone) != 0);
        pdone_mask = __ballot_sync(0xffffffffu, cnt > 0 && (flags & kStageParentDone) != 0);
    }
    if (rescan_mask) {  // chunks without records: find their fired particles again (tau < 0), in index order
        __syncthreads();  // (every warp is done with the list of the previous tile that needed one)
        for (int j = warp; j < CHUNKS; j += WARPS) {
            if (!((rescan_mask >> j) & 1u)) continue;
            const long long cbase = (first_chunk + j) * kChunk;
            unsigned int k = 0;
#pragma unroll
            for (int r4 = 0; r4 < kChunk / 32; ++r4) {
                const long long i = cbase + r4 * 32 + lane;
                const bool f = i < a.n && a.tau[i] < (TR)0;
                const unsigned int bal = __ballot_sync(0xffffffffu, f);
                if (f) list[j][k + __popc(bal & ((1u << lane) - 1u))] = (unsigned char)(r4 * 32 + lane);
                k += __popc(bal);
            }
        }
        __syncthreads();
    }
    for (unsigned int e0 = 0; e0 < total; e0 += THREADS) {
        const unsigned int e = e0 + tid;
        if (e0 + (unsigned)(tid & ~31) >= total) break;   // (the whole warp is past the tile's last event)
        // chunk of event e: the largest j with off_j <= e (ties are empty chunks followed by the one that holds
        // e; lanes past the last chunk carry off = total > e); the offsets live in the lanes' registers
        int j = 0;
#pragma unroll
        for (int step = 16; step > 0; step >>= 1) {
            const int cand = j + step;
            const unsigned int oc = __shfl_sync(0xffffffffu, off_lane, min(cand, 31));
            if (cand < 32 && oc <= e) j = cand;
        }
        const unsigned int off_j = __shfl_sync(0xffffffffu, off_lane, j);
        const long long slot = (long long)(slot_base + excl + e);
        if (e >= total) continue;
        const unsigned int r = e - off_j;
        const long long cbase = (first_chunk + j) * kChunk;
        if ((done_mask >> j) & 1u) {
            // the fused step generated this event already and rewrote its parent: move the secondaries to their slot
            typedef StepResult<R, TR, KIND> Res;
            const uint4* src = reinterpret_cast<const uint4*>(a.stage_rec + (first_chunk + j) * a.stage_stride + r * sizeof(Res));
            union { uint4 raw[sizeof(Res) / 16]; Res res; } u;
#pragma unroll
            for (int k = 0; k < (int)(sizeof(Res) / 16); ++k) u.raw[k] = __ldcs(src + k);
            const long long i = cbase + u.res.idx;
            if (slot < a.capacity) {
#pragma unroll
                for (int c = 0; c < (KIND == 0 ? 3 : 6); ++c) a.out_p[c][slot] = u.res.sec[c];
                a.out_tau[0][slot] = u.res.sec_tau[0];
                if (KIND == 1) a.out_tau[1][slot] = u.res.sec_tau[KIND == 1 ? 1 : 0];
                if (a.parent) a.parent[slot] = a.parent_base + i;
            } else {   // capacity rule (R16): parents beyond the capacity are left as the evolve pass left them
#pragma unroll
                for (int c = 0; c < 3; ++c) a.p[c][i] = u.res.old_p[c];
                a.tau[i] = u.res.tau_ev;
            }
            continue;
        }
        const bool pdone = (pdone_mask >> j) & 1u;
        if (slot >= a.capacity && !pdone) continue;  // capacity rule (R16): later parents untouched
        const bool staged = !((rescan_mask >> j) & 1u);
        double px, py, pz, c2;
        long long i;
        if (staged) {
            const uint4* src = reinterpret_cast<const uint4*>(
                a.stage_rec + (first_chunk + j) * a.stage_stride + r * StageRecord<R>::kBytes);
            union { uint4 raw[StageRecord<R>::kVecs]; StageRecord<R> rec; } u;
#pragma unroll
            for (int k = 0; k < StageRecord<R>::kVecs; ++k) u.raw[k] = __ldg(src + k);
            if (slot >= a.capacity) {   // (pdone) the evolve pass removed this photon already: put it back as it left it
                const long long ib = cbase + u.rec.idx;
#pragma unroll
                for (int c = 0; c < 3; ++c) a.p[c][ib] = u.rec.p[c];
                a.tau[ib] = (TR)u.rec.tau_ev;
                continue;
            }
            const double sp = a.units.p;
            px = u.rec.p[0] * sp; py = u.rec.p[1] * sp; pz = u.rec.p[2] * sp;   // (records hold the caller's units)
            c2 = u.rec.c2;
            i = cbase + u.rec.idx;
        } else {
            i = cbase + list[j][r];
            const double sp = a.units.p, se = a.units.e, sb = a.units.b;
            px = a.p[0][i] * sp; py = a.p[1][i] * sp; pz = a.p[2][i] * sp;
            c2 = event_c2<KIND>(px, py, pz, a.e[0][i] * se, a.e[1][i] * se, a.e[2][i] * se, a.b[0][i] * sb, a.b[1][i] * sb,
                                a.b[2][i] * sb);
        }
        const EventOut<R, TR> out = KIND == 0 ? qs_event_compute<R, TR>(a, i, px, py, pz, c2)
                                              : bw_event_compute<R, TR>(a, i, px, py, pz, c2);
        event_commit<R, TR, KIND>(a, i, slot, out, pdone);
    }
    }  // tiles
#undef PXQ_TILE_OF
}

}  // namespace pxq
