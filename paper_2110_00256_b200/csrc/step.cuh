// =====================================================================================
//  step.cuh -- the fused QED step (picsarqed_qed_step): one persistent, warp-specialised
//  kernel in which the evolve pass and the events of the
//  particles that fire (rows a5-a7, a9) run side by side on every SM.
//
//  Why: a parent that fired gets a new momentum and a new optical depth -- four scattered
//  8-byte stores.  Done in a second kernel, 0.25 ms after the evolve pass streamed those
//  sectors through L2, each store is a 32-byte read-modify-write in DRAM (282 of the 317 MB
//  the round-1 event pass moved).  Here the parents are rewritten a few microseconds after
//  their sectors were loaded, while they are still in L2: the stores merge there and the
//  sector goes back to DRAM once, whole.
//
//  An event is a chain of dependent L2 round trips (~16 000 cycles per warp pass measured inside
//  the loaded memory system), so hiding it takes many warps that do nothing but wait -- which costs
//  registers, the resource the evolve pass of evolve.cuh spends on loads in flight (80 of its 112
//  registers per thread hold data on its way from HBM).  So here the particle data travel by TMA
//  bulk copies (cp.async.bulk, completion on an mbarrier) into shared memory: bytes in flight cost no
//  registers, the streaming warps run in 64, and the register file has room for 12 event warps.
//
//  Roles inside a CTA (one CTA per SM):
//   * SW streaming warps.  A warp owns the 128 contiguous particles of a chunk per tile, in sub-chunks
//     of 16 bytes per lane and array (64 particles in fp64, 128 in fp32); NS sub-chunk stages per warp
//     in shared memory, refilled by the warp's lane 0 as soon as the warp has read them.  chi^2 in fp64
//     registers, table in shared memory, ballot/popc ranks as in evolve.cuh.  The records of the
//     particles that fired (momentum, chi^2, evolved tau, index in the chunk) go to a queue in shared
//     memory;
//   * (SW/4) groups of C event warps; a group serves four streaming warps.  Entry n of a streaming warp's
//     queue lives in buffer n % C and belongs to event warp n % C of the group, so every (queue, buffer)
//     pair has one producer and one consumer.  An event warp takes the next entry of each of its four
//     queues at a time, so that most lanes hold an event, samples it (Philox, guided search of eq.25/29,
//     eq.26/30), rewrites the parent in place and stores the secondaries as one array-of-structures
//     record in the chunk's segment of the staging buffer.
//  The placement of the secondaries in parent order needs the global prefix of the chunk
//  counts, which exists only when every chunk has been counted: tile_scan_kernel, then the
//  placement path of event_kernel (events.cuh) moves the staged secondaries to their slots
//  (a streaming copy) -- and undoes the parents beyond `capacity` (R16) from the
//  old values kept in the staged record.
// =====================================================================================
#pragma once
#include "qed_device.cuh"
#include "evolve.cuh"
#include "events.cuh"

namespace pxq {

constexpr int kStepGroup = 4;   // streaming warps served by one group of event warps

// what an event warp needs of a particle that fired (shared memory only)
template <typename R, typename TR> struct StepRecord;
template <> struct alignas(16) StepRecord<double, double> { double p[3]; double c2; double tau_ev; unsigned idx; unsigned pad; };
template <> struct alignas(16) StepRecord<float, double> { double c2; double tau_ev; float p[3]; unsigned idx; };
template <> struct alignas(16) StepRecord<float, float> { double c2; float p[3]; float tau_ev; unsigned idx; unsigned pad[3]; };

struct StepQueueHeader { long long chunk; unsigned total; unsigned pad; };

template <typename R, typename TR, int SPECIES>
struct StepArgs {
    EvolveArgs<R, TR> ev;       // arrays, table, rate_dt, stage_cnt, tile_sum, chunks_per_tile, units
    EventArgs<R, TR> ge;        // cdf table, seed, step, id_base, units (its arrays alias ev's, writable)
    unsigned char* stage_res;   // [n_chunks] segments (ev.stage_stride apart) of kStageCap StepResult<R, TR, SPECIES> --
                                // or StageRecord<R>, for the chunks a full queue sent to the record path of event_kernel
    int batch_wait;             // polls an event warp waits for a full batch (see the event warps' loop)
    int spill;                  // 1: a streaming warp that finds its queue buffer taken does not wait: the chunk goes to
                                // the record path of event_kernel (same routines, same results; its parents are then
                                // rewritten by scattered read-modify-writes)
};

__device__ __forceinline__ bool elect_one() {   // one lane of the (converged) warp
    unsigned pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
template <int N> __device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

__device__ __forceinline__ unsigned ld_flag(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"((unsigned)__cvta_generic_to_shared(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_flag(unsigned* p, unsigned v) {
    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(p)), "r"(v) : "memory");
}

// ---- TMA bulk copies global -> shared, completion counted in bytes on an mbarrier --------------------------
__device__ __forceinline__ void mbar_init(unsigned long long* mbar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(mbar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* mbar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                 ::"r"((unsigned)__cvta_generic_to_shared(mbar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* mbar, unsigned parity) {
    const unsigned mb = (unsigned)__cvta_generic_to_shared(mbar);
    unsigned done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(mb), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* mbar,
                                         unsigned long long policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "r"(bytes),
                   "r"((unsigned)__cvta_generic_to_shared(mbar)), "l"(policy) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "r"(bytes),
                   "r"((unsigned)__cvta_generic_to_shared(mbar)) : "memory");
}

// shared-memory layout of the kernel, after the table: [stages][record queues]
template <typename R, typename TR, int SW, int EW, int D, int NS>
struct StepLayout {
    static constexpr int V = 16 / sizeof(R);            // particles per lane and sub-chunk
    static constexpr int SUB = 32 * V;                  // particles per sub-chunk
    static constexpr int HALVES = kChunk / SUB;         // sub-chunks per chunk: 2 (fp64), 1 (fp32)
    static constexpr unsigned AB = SUB * sizeof(R);     // bytes of one array in a stage (512)
    static constexpr unsigned TB = SUB * sizeof(TR);
    static constexpr unsigned STAGE = 9 * AB + TB;
    static constexpr size_t stages_bytes = (size_t)SW * NS * STAGE;
    static constexpr size_t queue_bytes = (size_t)SW * D * kStageCap * sizeof(StepRecord<R, TR>);
    static constexpr int THREADS = (SW + EW) * 32;
    static constexpr int LAUNCH_REGS = ((65536 / THREADS) / 8) * 8;   // what __launch_bounds__(THREADS, 1) gives a thread
};

template <int N, int LAUNCH> __device__ __forceinline__ void reg_set() {   // N registers per thread from here on
    if constexpr (N > LAUNCH) reg_alloc<N>();
    else if constexpr (N > 0 && N < LAUNCH) reg_dealloc<N>();
}

// SW streaming warps (SW <= 32), EW event warps, D record buffers per streaming warp, NS sub-chunk stages per streaming warp.
// REG_S / REG_E: registers per thread of the two roles after setmaxnreg (0 = keep the launch allocation).
template <typename R, typename TR, int SPECIES, bool SCALED, int SW, int EW, int D, int NS, int REG_S, int REG_E>
__global__ void __launch_bounds__((SW + EW) * 32, 1) step_kernel(const StepArgs<R, TR, SPECIES> sa) {
    typedef StepLayout<R, TR, SW, EW, D, NS> L;
    constexpr int V = L::V, SUB = L::SUB, HALVES = L::HALVES;
    constexpr int TILE = SW * kChunk;
    static_assert(SW <= 32 && SW % 4 == 0 && EW % 4 == 0, "lane q of an event warp watches queue q; setmaxnreg acts on groups of four warps");
    typedef StepRecord<R, TR> Rec;
    typedef StepResult<R, TR, SPECIES> Res;
    const EvolveArgs<R, TR>& a = sa.ev;
    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // (a shuffle from lane 0: the compiler keeps it in a uniform register)
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned long long mbar;
    __shared__ unsigned long long full_bar[SW][NS];
    // queue of streaming warp q: entry n lives in buffer n % D.  produced[q] entries published (by q), claimed[q] entries
    // taken (compare-and-swap by the event warps), released[q][b] times buffer b has been handed back
    __shared__ unsigned produced[SW], claimed[SW], released[SW][D], finished[SW];
    __shared__ StepQueueHeader header[SW][D];

    const R* tab = a.tab.L;
    if (a.table_in_smem) {
        const unsigned bytes = ((unsigned)(a.tab.n * sizeof(R)) + 15u) & ~15u;
        stage_table_tma(smem_raw, a.tab.L, bytes, &mbar);
        tab = reinterpret_cast<const R*>(smem_raw);
    }
    if (threadIdx.x < SW) {
        finished[threadIdx.x] = produced[threadIdx.x] = claimed[threadIdx.x] = 0u;
        for (int b = 0; b < D; ++b) released[threadIdx.x][b] = 0u;
        for (int s = 0; s < NS; ++s) mbar_init(&full_bar[threadIdx.x][s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned char* const stages = smem_raw + a.table_bytes;
    Rec* const recs = reinterpret_cast<Rec*>(stages + L::stages_bytes);   // [SW][D][kStageCap]
    const long long ntiles_full = a.n / TILE;

    if (warp < SW) {
        // ================================ streaming warps =========================================
        reg_set<REG_S, L::LAUNCH_REGS>();
        const unsigned long long pol_stream = l2_policy_evict_first();
        // this warp's sequence of sub-chunks: j = 0, 1, ...; tile blockIdx.x + (j / HALVES) gridDim.x, half j % HALVES
        const long long my_tiles = ntiles_full > blockIdx.x ? (ntiles_full - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
        const long long n_sub = my_tiles * HALVES;
        unsigned char* const my_stages = stages + (size_t)warp * NS * L::STAGE;
        auto sub_base = [&](long long j) -> long long {
            const long long tile = blockIdx.x + (j / HALVES) * gridDim.x;
            return tile * TILE + (long long)warp * kChunk + (j % HALVES) * SUB;
        };
        auto issue = [&](long long j) {   // (all lanes call it) sub-chunk j -> stage j % NS: ten bulk copies by one elected lane
            const int s = (int)(j % NS);
            unsigned char* dst = my_stages + (size_t)s * L::STAGE;
            const long long i0 = sub_base(j);
            if (elect_one()) {
                mbar_expect_tx(&full_bar[warp][s], L::STAGE);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    // (momenta and tau: no eviction hint, they are rewritten by this kernel and should outlive the fields in L2)
                    bulk_g2s(dst + c * L::AB, a.p[c] + i0, L::AB, &full_bar[warp][s]);
                    bulk_g2s(dst + (3 + c) * L::AB, a.e[c] + i0, L::AB, &full_bar[warp][s], pol_stream);
                    bulk_g2s(dst + (6 + c) * L::AB, a.b[c] + i0, L::AB, &full_bar[warp][s], pol_stream);
                }
                bulk_g2s(dst + 9 * L::AB, a.tau + i0, L::TB, &full_bar[warp][s]);
            }
        };
        for (long long j = 0; j < NS && j < n_sub; ++j) issue(j);
        unsigned n_pub = 0;                       // entries this warp has published
        unsigned total = 0;                       // fired particles of the current chunk so far (over its sub-chunks)
        bool queued = false, spilled = false, have_buf = false;
        Rec* wbuf = nullptr;
        for (long long j = 0; j < n_sub; ++j) {
            const int s = (int)(j % NS);
            const int half = (int)(j % HALVES);
            const long long base = sub_base(j);
            const long long chunk = (base - half * SUB) / kChunk;
            mbar_wait(&full_bar[warp][s], (unsigned)((j / NS) & 1));
            const unsigned char* st = my_stages + (size_t)s * L::STAGE;
            Vec<R, V> q[9];
#pragma unroll
            for (int c = 0; c < 9; ++c) q[c] = *reinterpret_cast<const Vec<R, V>*>(st + c * L::AB + lane * 16);
            Vec<TR, V> t = *reinterpret_cast<const Vec<TR, V>*>(st + 9 * L::AB + lane * (V * sizeof(TR)));
            // every lane has read the stage: refill it (the bulk copy lands a DRAM round trip from now, long after the
            // shared-memory loads above have returned)
            __syncwarp();
            if (j + NS < n_sub) issue(j + NS);
            unsigned int fired_bits = 0;
            double c2s[V];
            {
                R in[9][V], d[V];
#pragma unroll
                for (int c = 0; c < 9; ++c)
#pragma unroll
                    for (int v = 0; v < V; ++v) in[c][v] = q[c].v[v];
                decrement_vec<R, SPECIES, SCALED, V>(in, tab, a.tab, a.rate_dt, a.units, d, c2s);
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    const TR tn = t.v[v] - (TR)d[v];
                    t.v[v] = tn;
                    if (tn < (TR)0) fired_bits |= 1u << v;
                }
            }
            // rank inside the chunk, in index order (sub-chunk, lane, v): ballot / popc
            const unsigned int lt = (1u << lane) - 1u;
            unsigned int below = 0, all = 0;
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const unsigned int bal = __ballot_sync(0xffffffffu, (fired_bits >> v) & 1u);
                below += __popc(bal & lt);
                all += __popc(bal);
            }
            if (half == 0) { total = 0; queued = true; spilled = false; have_buf = false; }
            unsigned int r = total + below;
            total += all;
            // the evolved tau goes out BEFORE the chunk is published: the event warp's store of the new tau must land on top
            st_vec<TR, V>(a.tau + base + lane * V, t);
            if (all > 0 && queued && !spilled && !have_buf) {
                // the first records of the chunk: take buffer n_pub % D of this warp's queue (free when entry n_pub - D
                // has been handed back)
                const unsigned b = n_pub % D, k = n_pub / D;
                auto room = [&]() {
                    unsigned e = 0;
                    if (lane == 0) e = ld_flag(&released[warp][b]);
                    return __shfl_sync(0xffffffffu, e, 0) == k;
                };
                if (sa.spill) {
                    if (!room()) spilled = true;
                } else {
                    while (!room()) __nanosleep(64);
                }
                wbuf = recs + ((size_t)warp * D + b) * kStageCap;
                have_buf = !spilled;
            }
            if (total > (unsigned)kStageCap) queued = false;   // too many for a segment: the re-scan path of event_kernel
            if (all > 0 && queued) {
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    if ((fired_bits >> v) & 1u) {
                        const unsigned idx = (unsigned)(half * SUB + lane * V + v);
                        if (!spilled) {
                            Rec& rec = wbuf[r];
                            rec.p[0] = q[0].v[v];
                            rec.p[1] = q[1].v[v];
                            rec.p[2] = q[2].v[v];
                            rec.c2 = c2s[v];
                            rec.tau_ev = t.v[v];
                            rec.idx = idx;
                        } else {   // (rare) straight to the chunk's segment in global memory, as a StageRecord
                            StageRecord<R>* g = reinterpret_cast<StageRecord<R>*>(sa.stage_res + chunk * a.stage_stride) + r;
                            g->p[0] = q[0].v[v];
                            g->p[1] = q[1].v[v];
                            g->p[2] = q[2].v[v];
                            g->c2 = c2s[v];
                            g->idx = idx;
                            g->tau_ev = (double)t.v[v];
                        }
                        ++r;
                    }
                }
            }
            if (half == HALVES - 1) {   // the chunk is complete
                const bool publish = total > 0 && queued && !spilled;
                if (lane == 0) {
                    a.stage_cnt[chunk] = (unsigned short)(total == 0 ? 0u : (publish ? (total | kStageDone)
                                                                                    : (queued ? total : (total | kStageNoRecords))));
                    if (total > 0) atomicAdd(a.tile_sum + chunk / kEventTileChunks, total);
                    if (publish) {
                        header[warp][n_pub % D].chunk = chunk;
                        header[warp][n_pub % D].total = total;
                    }
                }
                if (publish) {
                    __syncwarp();
                    ++n_pub;
                    if (lane == 0) st_flag(&produced[warp], n_pub);   // release: records, header, tau stores
                }
            }
        }
        // ragged last tile: scalar, guarded; it stages nothing (its chunks are counted from tau afterwards and take the
        // re-scan path of event_kernel)
        if (blockIdx.x == (unsigned)(ntiles_full % gridDim.x)) {
            for (long long i = ntiles_full * TILE + warp * 32 + lane; i < a.n; i += SW * 32) {
                const R d = decrement_one<R, SPECIES, SCALED>(a.p[0][i], a.p[1][i], a.p[2][i], a.e[0][i], a.e[1][i], a.e[2][i],
                                                              a.b[0][i], a.b[1][i], a.b[2][i], tab, a.tab, a.rate_dt, a.units);
                a.tau[i] = a.tau[i] - (TR)d;
            }
        }
        __syncwarp();
        if (lane == 0) st_flag(&finished[warp], 1u);
    } else {
        // ================================ event warps ============================================
        reg_set<REG_E, L::LAUNCH_REGS>();
        const EventArgs<R, TR>& g = sa.ge;
        const int ew = warp - SW;
        int idle_polls = 0;
        unsigned rot = (unsigned)(ew * 4) % SW;   // where this warp starts looking (spreads the event warps over the queues)
        while (true) {
            // lane q < SW looks at queue q
            unsigned avail = 0, fin = 1, my_claim = 0;
            if (lane < SW) {
                fin = ld_flag(&finished[lane]);                         // (read before `produced`: a finished queue is final)
                my_claim = *reinterpret_cast<volatile unsigned*>(&claimed[lane]);
                const unsigned prod = ld_flag(&produced[lane]);
                avail = prod != my_claim ? 1u : 0u;
                if (avail) fin = 0;
            }
            const unsigned avail_mask = __ballot_sync(0xffffffffu, avail != 0);
            // A pass costs the same instructions whether 5 or 32 lanes hold an event, and the kernel is bound by instruction
            // issue: wait for four chunks (about 31 events) unless the queues are running dry.
            if (avail_mask == 0 || (__popc(avail_mask) < 4 && idle_polls < sa.batch_wait)) {
                if (avail_mask == 0 && __all_sync(0xffffffffu, fin != 0)) break;
                ++idle_polls;
                __nanosleep(2000);   // (a poll costs issue slots the streaming warps need; a chunk arrives every few microseconds)
                continue;
            }
            idle_polls = 0;
            // take up to four queues, first come from `rot` on, and claim their next entry (another event warp may be
            // quicker: up to three rounds over what is left)
            constexpr unsigned kAll = (SW == 32) ? 0xffffffffu : ((1u << SW) - 1u);
            unsigned left = ((avail_mask >> rot) | (avail_mask << (SW - rot))) & kAll;   // bit k: queue (rot + k) % SW
            unsigned got_mask = 0;
            bool got = false;
            for (int round = 0; round < 3 && left != 0 && __popc(got_mask) < 4; ++round) {
                unsigned pick = 0;
                const int need = 4 - __popc(got_mask);
                for (int k = 0; k < need && left != 0; ++k) {
                    const unsigned low = left & (0u - left);
                    pick |= low;
                    left ^= low;
                }
                const unsigned pick_mask = ((pick << rot) | (pick >> (SW - rot))) & kAll;
                bool ok = false;
                if ((pick_mask >> lane) & 1u) ok = atomicCAS(&claimed[lane], my_claim, my_claim + 1u) == my_claim;
                got = got || ok;
                got_mask |= __ballot_sync(0xffffffffu, ok);
            }
            rot = (rot + 5) % SW;
            if (got_mask == 0) continue;
            unsigned cnt_src = 0;
            long long chunk_src = 0;
            if (got) {
                const StepQueueHeader h = header[lane][my_claim % D];
                cnt_src = h.total;
                chunk_src = h.chunk;
            }
            // lanes 0..3 take over the (at most four) entries of the batch, in queue order
            const int n_got = __popc(got_mask);
            const int src = lane < n_got ? (int)__fns(got_mask, 0, lane + 1) : 0;
            unsigned cnt = __shfl_sync(0xffffffffu, cnt_src, src);
            const long long chunk_l = __shfl_sync(0xffffffffu, chunk_src, src);
            const unsigned entry_l = __shfl_sync(0xffffffffu, my_claim, src);
            if (lane >= n_got) cnt = 0;
            const int q_l = src;
            unsigned incl = cnt;   // offsets of the chunks of this batch
#pragma unroll
            for (int d = 1; d < 4; d <<= 1) {
                const unsigned o = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += o;
            }
            const unsigned off_l = incl - cnt;
            const unsigned total = __shfl_sync(0xffffffffu, incl, 3);
            for (unsigned e0 = 0; e0 < total; e0 += 32) {
                const unsigned e = e0 + lane;
                int j = 0;
#pragma unroll
                for (int k = 1; k < 4; ++k) {
                    const unsigned ok = __shfl_sync(0xffffffffu, off_l, k);
                    const unsigned ck = __shfl_sync(0xffffffffu, cnt, k);
                    if (ck > 0 && ok <= e) j = k;
                }
                const unsigned off_j = __shfl_sync(0xffffffffu, off_l, j);
                const long long chunk = __shfl_sync(0xffffffffu, chunk_l, j);
                const unsigned entry = __shfl_sync(0xffffffffu, entry_l, j);
                const int q = __shfl_sync(0xffffffffu, q_l, j);
                if (e >= total) continue;
                const unsigned r = e - off_j;
                const Rec rec = recs[((size_t)q * D + entry % D) * kStageCap + r];
                const long long i = chunk * kChunk + rec.idx;
                const double sp = g.units.p;
                const double px = rec.p[0] * sp, py = rec.p[1] * sp, pz = rec.p[2] * sp;
                const EventOut<R, TR> out = SPECIES == 0 ? qs_event_compute<R, TR>(g, i, px, py, pz, rec.c2)
                                                         : bw_event_compute<R, TR>(g, i, px, py, pz, rec.c2);
                // the parent, in place: its sectors were loaded a few microseconds ago and are still in L2
#pragma unroll
                for (int c = 0; c < 3; ++c) g.p[c][i] = out.parent_p[c];
                g.tau[i] = out.parent_tau;
                // the secondaries (and what undoes the parent if the output turns out to be full): one record
                union { Res res; uint4 raw[sizeof(Res) / 16]; } o;
#pragma unroll
                for (int c = 0; c < (SPECIES == 0 ? 3 : 6); ++c) o.res.sec[c] = out.sec[c];
                o.res.sec_tau[0] = out.sec_tau[0];
                if (SPECIES == 1) o.res.sec_tau[SPECIES == 1 ? 1 : 0] = out.sec_tau[1];
#pragma unroll
                for (int c = 0; c < 3; ++c) o.res.old_p[c] = rec.p[c];
                o.res.tau_ev = rec.tau_ev;
                o.res.idx = rec.idx;
                uint4* dst = reinterpret_cast<uint4*>(sa.stage_res + chunk * a.stage_stride + r * sizeof(Res));
#pragma unroll
                for (int k = 0; k < (int)(sizeof(Res) / 16); ++k) dst[k] = o.raw[k];
            }
            __syncwarp();
            if (lane < n_got) st_flag(&released[q_l][entry_l % D], entry_l / D + 1u);   // release: the buffer may be overwritten
        }
    }
}

}  // namespace pxq
