// =====================================================================================
//  picsarqed.cu -- the C ABI of include/picsarqed.h: context, table storage, launchers.
//  Compiled only for sm_100a.  No CPU fallback: every entry point enqueues CUDA kernels.
// =====================================================================================
#include "../../include/picsarqed.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "evolve.cuh"
#include "events.cuh"
#include "tables.cuh"
#include "cascade.cuh"
#include "lookup.cuh"
#include "step.cuh"

using namespace pxq;

constexpr int kMaxSlabs = 64;

struct picsarqed_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 0;
    std::string err;

    bool have_tables = false;
    picsarqed_table_params tp{};
    double* tab64[4] = {nullptr, nullptr, nullptr, nullptr};  // lnG, qs_lnP, lnT, bw_P
    float* tab32[4] = {nullptr, nullptr, nullptr, nullptr};   // fp32-rounded copies
    size_t tab_n[4] = {0, 0, 0, 0};
    // search guides of the two CDF tables (see Table2D::guide), [0] photon emission, [1] pair production
    unsigned short* guide[2] = {nullptr, nullptr};
    size_t guide_bytes[2] = {0, 0};
    double guide_k0[2] = {0.0, 0.0}, guide_inv_dk[2] = {0.0, 0.0};
    double* d_scalar = nullptr;

    // evolve: per-CTA counts + arrival ticket
    unsigned int* partials = nullptr;
    unsigned int* ticket = nullptr;
    int partials_cap = 0;
    // tuning knobs (picsarqed_set_option)
    int evolve_unroll = 0;       // 0 = default per dtype
    int evolve_ctas_per_sm = 0;  // 0 = occupancy
    // unit system of the caller's arrays (picsarqed_set_units): multipliers to p/(m_e c), E/E_s, cB/E_s, seconds
    UnitScales units;
    double t_scale = 1.0;
    int unit_system = 0;
    int event_config = 0;        // shape of event_kernel: see launch_event_pass
    int fused_step = 0;          // qed_step: 1 = the warp-specialised fused kernel (step.cuh), 0 = evolve pass + event pass
    // "stage_records" = 1: evolve_optical_depth also stages the records of the particles that fire, and a generate_photons
    // / generate_pairs call that follows ON THE SAME ARRAYS (the caller's promise: momenta, fields and tau untouched in
    // between) takes them instead of re-scanning tau and gathering the parents
    int stage_records = 0;
    bool staged_valid = false;
    const void* staged_tau = nullptr;
    long long staged_n = 0;
    int staged_species = -1, staged_dtype = -1, staged_tau_dtype = -1;
    double chi_event_min = 0.0;   // PAPER.md:340 (picsarqed_set_chi_threshold): no event below it; 0 = off
    int step_spill = 0;          // fused kernel: 1 = a streaming warp whose queue is full hands the chunk to the record path
    int step_batch_wait = 0;     // fused kernel: polls (2 us each) an event warp waits for four chunks before it takes fewer
    int step_config = 0;         // fused kernel: see launch_fused_step
    int evolve_redraw = 2;       // qed_step of leptons: see launch_step
    int event_pdl = 1;           // the event kernel is launched as a programmatic dependent of the offsets scan
    int time_kernels = 0;        // qed_step brackets its evolve pass and its event pass with CUDA events
    std::vector<cudaEvent_t> timing_events;  // triples (start, after evolve, after events), not yet read
    // per-chunk scratch of the event path: staged records, counts, output offsets (see events.cuh)
    void* rec = nullptr;
    size_t rec_bytes = 0;
    size_t rec_sum_bytes = 0;  // its first bytes: the tile sums
    // host-path staging
    void* stage = nullptr;
    size_t stage_bytes = 0;
    // step_host pipeline: slab k is copied in on h2d_stream, stepped on stream, copied out on d2h_stream;
    // d_counts[k] = events of the slabs before slab k (d_counts[0] = 0), so the secondaries of all slabs land
    // densely, in parent order, in one buffer
    unsigned long long* d_counts = nullptr;  // kMaxSlabs + 2 device counters
    unsigned long long* h_counts = nullptr;  // pinned copy of d_counts
    cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
    std::vector<cudaEvent_t> slab_events;    // 2 per slab: copied in, stepped
    int host_slabs = 0;                      // 0 = automatic, k = split step_host into (at most) k slabs
    const unsigned long long* link_slot_base = nullptr;  // set by step_host around the qed_step of a slab
    long long link_parent_base = 0;
    // closed loop (cascade_step): constant field arrays + secondary buffers, device counters and their pinned copy
    void* cas = nullptr;
    size_t cas_bytes = 0;
    long long cas_field_n = 0;          // entries of the six field arrays that hold cas_field[]
    double cas_field[6] = {0, 0, 0, 0, 0, 0};
    int cas_field_dtype = -1;
    unsigned long long* d_cas = nullptr;  // 16 counters
    unsigned long long* h_cas = nullptr;
    double build_ms = 0.0;
    cudaStream_t aux_stream = nullptr;       // build_tables: the second process
    cudaEvent_t aux_event[2] = {nullptr, nullptr};
    cudaEvent_t build_event[2] = {nullptr, nullptr};   // around the quadrature kernels of the last build_tables
};

namespace {

int fail(picsarqed_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg;
    return code;
}
#define PXQ_CUDA(ctx, call)                                                                      \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess)                                                                   \
            return fail(ctx, PICSARQED_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// rows of the 2D tables (0 in the params = the 1D count)
int rows_2d(const picsarqed_table_params& p, int kind) {
    const int r = kind == 0 ? p.qs_n_chi_2d : p.bw_n_chi_2d;
    return r > 0 ? r : (kind == 0 ? p.qs_n_chi : p.bw_n_chi);
}

bool params_ok(const picsarqed_table_params* p) {
    return p && (p->qs_n_chi_2d == 0 || p->qs_n_chi_2d >= 2) && (p->bw_n_chi_2d == 0 || p->bw_n_chi_2d >= 2) && p->qs_n_chi >= 2 && p->qs_n_xi >= 2 && p->bw_n_chi >= 2 && p->bw_n_xi >= 2 &&
           p->qs_chi_min > 0 && p->qs_chi_max > p->qs_chi_min && p->bw_chi_min > 0 &&
           p->bw_chi_max > p->bw_chi_min && p->qs_xi_min > 0 && p->qs_xi_min < 1;
}

void table_sizes(const picsarqed_table_params& p, size_t n[4]) {
    n[0] = (size_t)p.qs_n_chi;
    n[1] = (size_t)rows_2d(p, 0) * p.qs_n_xi;
    n[2] = (size_t)p.bw_n_chi;
    n[3] = (size_t)rows_2d(p, 1) * p.bw_n_xi;
}

__global__ void narrow_kernel(const double* __restrict__ src, float* __restrict__ dst, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = (float)src[i];
}

// elements of zero padding behind every table: 16-byte TMA copies of the 1D tables and the unconditional column loads of
// search_row's fast path (kGuideFastSpan columns past the bracket) stay in bounds
constexpr size_t kTablePad = 16;

// (re)allocate table storage for params p; +2 elements of padding so that 16-byte TMA copies stay in bounds
int alloc_tables(picsarqed_ctx* c, const picsarqed_table_params& p) {
    size_t n[4];
    table_sizes(p, n);
    for (int k = 0; k < 4; ++k) {
        if (c->tab_n[k] != n[k] || !c->tab64[k] || !c->tab32[k]) {   // (a rebuild of the same geometry keeps its buffers)
            if (c->tab64[k]) cudaFree(c->tab64[k]);
            if (c->tab32[k]) cudaFree(c->tab32[k]);
            c->tab64[k] = nullptr;
            c->tab32[k] = nullptr;
            c->tab_n[k] = 0;
            PXQ_CUDA(c, cudaMalloc(&c->tab64[k], (n[k] + kTablePad) * sizeof(double)));
            PXQ_CUDA(c, cudaMalloc(&c->tab32[k], (n[k] + kTablePad) * sizeof(float)));
        }
        PXQ_CUDA(c, cudaMemsetAsync(c->tab64[k], 0, (n[k] + kTablePad) * sizeof(double), c->stream));
        PXQ_CUDA(c, cudaMemsetAsync(c->tab32[k], 0, (n[k] + kTablePad) * sizeof(float), c->stream));
        c->tab_n[k] = n[k];
    }
    c->tp = p;
    return PICSARQED_OK;
}

int narrow_tables(picsarqed_ctx* c) {
    for (int k = 0; k < 4; ++k) {
        const size_t n = c->tab_n[k];
        const int grid = (int)std::min<size_t>((n + 255) / 256, 1184);
        narrow_kernel<<<grid, 256, 0, c->stream>>>(c->tab64[k], c->tab32[k], n);
    }
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

constexpr int kGuideBins = 2048;   // measured: 256 -> 1024 -> 2048 -> 4096 bins: config 5 event passes 1.77 -> 1.63 -> 1.58 -> 1.55 ms

// minimum of column 0 over the rows (lower end of the key range of the photon-emission guide)
__global__ void column0_min_kernel(const double* __restrict__ tab, int n_rows, int n_cols, double* out) {
    __shared__ double red[256];
    double m = INFINITY;
    for (int r = threadIdx.x; r < n_rows; r += blockDim.x) m = fmin(m, tab[(size_t)r * n_cols]);
    red[threadIdx.x] = m;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) red[threadIdx.x] = fmin(red[threadIdx.x], red[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = red[0];
}

// guide[n][j] = max{m : tab[n][m] <= key_j}, 0 if there is none and for j = 0 (whose lower edge is -inf).
// split = 0 (pair production: the table holds P, the key is r'): key_j = k0 + j dk.
// split = 1 (photon emission: the table holds ln P, the key is ln r): the lower half of the bins is uniform in ln r on [k0, ln 1/2]
// (dk = its spacing), the upper half uniform in r on [1/2, 1] -- with all bins uniform in ln r the last one, ln r in [-dk, 0], holds
// the whole flat end of a low-chi row (hundreds of columns) and is hit by 0.5-1 % of the events: a quarter of the warps
__global__ void guide_kernel(const double* __restrict__ tab, int n_rows, int n_cols, double k0, double dk, int bins, int split,
                             unsigned short* __restrict__ guide) {
    const long long total = (long long)n_rows * (bins + 1);
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(t / (bins + 1)), j = (int)(t % (bins + 1));
        double key = k0 + j * dk;
        if (split && j >= bins / 2) key = j == bins ? 0.0 : log(0.5 + (j - bins / 2) * (0.5 / (bins / 2)));
        const double* row = tab + (size_t)n * n_cols;
        int lo = -1, hi = n_cols;  // row[lo] <= key < row[hi]
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (row[mid] <= key) lo = mid; else hi = mid;
        }
        guide[t] = (unsigned short)(j == 0 ? 0 : max(lo, 0));
    }
}

int build_guides(picsarqed_ctx* c) {
    for (int kind = 0; kind < 2; ++kind) {
        const int rows = rows_2d(c->tp, kind), cols = kind == 0 ? c->tp.qs_n_xi : c->tp.bw_n_xi;
        const size_t want = (size_t)rows * (kGuideBins + 1) * sizeof(unsigned short);
        if (c->guide[kind] && c->guide_bytes[kind] != want) {   // (a rebuild of the same geometry keeps its buffer)
            cudaFree(c->guide[kind]);
            c->guide[kind] = nullptr;
        }
        unsigned short* keep = c->guide[kind];
        c->guide[kind] = nullptr;                                // (no guide while it is being rebuilt, or if it cannot be built)
        auto drop = [&]() { if (keep) cudaFree(keep); keep = nullptr; c->guide_bytes[kind] = 0; };
        if (cols > 65535) { drop(); continue; }  // indices are stored in 16 bits; wider tables are searched unguided
        const double* tab = c->tab64[kind == 0 ? PICSARQED_TAB_QS_LNP : PICSARQED_TAB_BW_P];
        double k0 = 0.0, k1 = 0.5;
        if (kind == 0) {
            if (!c->d_scalar) PXQ_CUDA(c, cudaMalloc(&c->d_scalar, sizeof(double)));
            column0_min_kernel<<<1, 256, 0, c->stream>>>(tab, rows, cols, c->d_scalar);
            PXQ_CUDA(c, cudaMemcpyAsync(&k0, c->d_scalar, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
            k1 = std::log(0.5);
            if (!std::isfinite(k0) || !(k0 < k1)) { drop(); continue; }
        }
        // (photon emission: the lower half of the bins covers [k0, ln 1/2] uniformly in ln r, the upper half [1/2, 1] uniformly in r)
        const double dk = (k1 - k0) / (kind == 0 ? kGuideBins / 2 : kGuideBins);
        if (!keep) PXQ_CUDA(c, cudaMalloc(&keep, want));
        c->guide_bytes[kind] = want;
        c->guide[kind] = keep;
        guide_kernel<<<c->num_sms * 4, 256, 0, c->stream>>>(tab, rows, cols, k0, dk, kGuideBins, kind == 0 ? 1 : 0, c->guide[kind]);
        PXQ_CUDA(c, cudaGetLastError());
        c->guide_k0[kind] = k0;
        c->guide_inv_dk[kind] = 1.0 / dk;
    }
    return PICSARQED_OK;
}

template <typename R> const R* table_ptr(const picsarqed_ctx* c, int which);
template <> const double* table_ptr<double>(const picsarqed_ctx* c, int which) { return c->tab64[which]; }
template <> const float* table_ptr<float>(const picsarqed_ctx* c, int which) { return c->tab32[which]; }

template <typename R>
Table1D<R> view_1d(const picsarqed_ctx* c, int species) {
    Table1D<R> t;
    const auto& p = c->tp;
    const double lo = species == 0 ? p.qs_chi_min : p.bw_chi_min, hi = species == 0 ? p.qs_chi_max : p.bw_chi_max;
    t.n = species == 0 ? p.qs_n_chi : p.bw_n_chi;
    t.L = table_ptr<R>(c, species == 0 ? PICSARQED_TAB_LNG : PICSARQED_TAB_LNT);
    t.ln_min = std::log(lo);
    t.ln_max = std::log(hi);
    t.inv_delta = (t.n - 1) / (t.ln_max - t.ln_min);
    t.chi_min = lo;
    t.chi_max = hi;
    t.c2_event_min = c->chi_event_min * c->chi_event_min;
    return t;
}

template <typename R>
Table2D<R> view_2d(const picsarqed_ctx* c, int species) {
    Table2D<R> t;
    const auto& p = c->tp;
    const double lo = species == 0 ? p.qs_chi_min : p.bw_chi_min, hi = species == 0 ? p.qs_chi_max : p.bw_chi_max;
    t.n_chi = rows_2d(p, species);
    t.n_xi = species == 0 ? p.qs_n_xi : p.bw_n_xi;
    t.P = table_ptr<R>(c, species == 0 ? PICSARQED_TAB_QS_LNP : PICSARQED_TAB_BW_P);
    t.ln_min = std::log(lo);
    t.ln_max = std::log(hi);
    t.inv_delta = (t.n_chi - 1) / (t.ln_max - t.ln_min);
    t.ln_xi_min = species == 0 ? std::log(p.qs_xi_min) : 0.0;
    t.xi_step = species == 0 ? -t.ln_xi_min / (double)(t.n_xi - 1) : 0.5 / (double)(t.n_xi - 1);
    t.guide = c->guide[species];
    t.guide_bins = kGuideBins;
    t.guide_split = species == 0 ? 1 : 0;
    t.guide_k0 = c->guide_k0[species];
    t.guide_inv_dk = c->guide_inv_dk[species];
    return t;
}

// ---- the scratch of picsarqed_generate_photons_noalloc (include/picsarqed.h): chunk counts, tile offsets, tile sums
// of up to kNoAllocMaxN particles, laid out as chunk_scratch lays them out, in a file-scope device array that every
// GPU which loads the library holds until exit.  In host code the array's NAME is a host-side stand-in, not a device
// address: the address a kernel can use comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr long long kNoAllocMaxN = 1ll << 24;
constexpr long long kNoAllocChunks = kNoAllocMaxN / kChunk;
constexpr size_t kNoAllocSumBytes = ((size_t)(kNoAllocChunks / 8 + 2) * sizeof(unsigned int) + 255) & ~(size_t)255;
constexpr size_t kNoAllocCntBytes = ((size_t)kNoAllocChunks * sizeof(unsigned short) + 255) & ~(size_t)255;
constexpr size_t kNoAllocOffBytes = ((size_t)(kNoAllocChunks / 8 + 2) * sizeof(unsigned long long) + 255) & ~(size_t)255;
constexpr size_t kNoAllocBytes = kNoAllocSumBytes + kNoAllocCntBytes + kNoAllocOffBytes;   // 459 264 bytes
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
void* g_noalloc_ptr[kNoAllocMaxDevices] = {};

// the device address of g_noalloc_scratch on `device`, which must be the current device
cudaError_t noalloc_scratch_address(int device, void** out) {
    *out = nullptr;
    if (device < 0 || device >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[device]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_noalloc_ptr[device] = ptr;
    }
    *out = g_noalloc_ptr[device];
    return cudaSuccess;
}

}  // namespace

// =====================================================================================
//  context and tables
// =====================================================================================
extern "C" {

int picsarqed_version(void) {
    int rt = 0;
    cudaRuntimeGetVersion(&rt);
    return (rt << 1) | 1;
}

int picsarqed_create(picsarqed_ctx** out, int cuda_device, void* cuda_stream) {
    if (!out) return PICSARQED_ERR_INVALID;
    *out = nullptr;
    picsarqed_ctx* c = new (std::nothrow) picsarqed_ctx();
    if (!c) return PICSARQED_ERR_CUDA;
    c->device = cuda_device;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    cudaError_t e = cudaSetDevice(cuda_device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cuda_device);
    if (e == cudaSuccess && prop.major != 10) {
        delete c;
        return PICSARQED_ERR_CUDA;  // built for sm_100a only; no fallback path
    }
    if (e == cudaSuccess) {
        c->num_sms = prop.multiProcessorCount;
        c->partials_cap = c->num_sms * 32;
        e = cudaMalloc(&c->partials, c->partials_cap * sizeof(unsigned int));
    }
    if (e == cudaSuccess) e = cudaMalloc(&c->ticket, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(c->ticket, 0, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_counts, (kMaxSlabs + 2) * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_counts, (kMaxSlabs + 2) * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc(&c->d_cas, 16 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_cas, 16 * sizeof(unsigned long long));
    if (e != cudaSuccess) {
        picsarqed_destroy(c);   // (frees whatever was allocated: every pointer starts as NULL)
        return PICSARQED_ERR_CUDA;
    }
    *out = c;
    {   // set-up of the no-alloc entry point: the device is current here (a failure is reported by that entry point)
        void* scratch = nullptr;
        (void)noalloc_scratch_address(cuda_device, &scratch);
    }
    // PICSARQED_OPTIONS="name=value,name=value": set_option calls applied to every new context (tuning experiments)
    if (const char* env = std::getenv("PICSARQED_OPTIONS")) {
        std::string all(env);
        size_t pos = 0;
        while (pos < all.size()) {
            const size_t end = all.find(',', pos);
            const std::string item = all.substr(pos, end == std::string::npos ? std::string::npos : end - pos);
            const size_t eq = item.find('=');
            if (eq != std::string::npos) picsarqed_set_option(c, item.substr(0, eq).c_str(), std::atoll(item.c_str() + eq + 1));
            if (end == std::string::npos) break;
            pos = end + 1;
        }
    }
    return PICSARQED_OK;
}

int picsarqed_destroy(picsarqed_ctx* c) {
    if (!c) return PICSARQED_ERR_INVALID;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    for (int k = 0; k < 4; ++k) {
        cudaFree(c->tab64[k]);
        cudaFree(c->tab32[k]);
    }
    cudaFree(c->partials);
    cudaFree(c->ticket);
    cudaFree(c->stage);
    cudaFree(c->rec);
    cudaFree(c->guide[0]);
    cudaFree(c->guide[1]);
    cudaFree(c->d_scalar);
    for (cudaEvent_t e : c->timing_events) cudaEventDestroy(e);
    cudaFree(c->d_counts);
    cudaFreeHost(c->h_counts);
    cudaFree(c->cas);
    cudaFree(c->d_cas);
    cudaFreeHost(c->h_cas);
    for (cudaEvent_t e : c->slab_events) cudaEventDestroy(e);
    if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
    for (int k = 0; k < 2; ++k) if (c->aux_event[k]) cudaEventDestroy(c->aux_event[k]);
    for (int k = 0; k < 2; ++k) if (c->build_event[k]) cudaEventDestroy(c->build_event[k]);
    if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
    if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
    delete c;
    return PICSARQED_OK;
}

const char* picsarqed_last_error(const picsarqed_ctx* c) { return c ? c->err.c_str() : "null context"; }

int picsarqed_set_option(picsarqed_ctx* c, const char* name, long long value) {
    if (!c || !name) return PICSARQED_ERR_INVALID;
    if (!std::strcmp(name, "evolve_unroll") && (value == 0 || value == 1 || value == 2 || value == 4))
        c->evolve_unroll = (int)value;
    else if (!std::strcmp(name, "evolve_ctas_per_sm") && value >= 0 && value <= 32)
        c->evolve_ctas_per_sm = (int)value;
    else if (!std::strcmp(name, "time_kernels") && (value == 0 || value == 1))
        c->time_kernels = (int)value;
    else if (!std::strcmp(name, "event_config") && value >= 0 && value <= 1)
        c->event_config = (int)value;
    else if (!std::strcmp(name, "fused_step") && (value == 0 || value == 1))
        c->fused_step = (int)value;
    else if (!std::strcmp(name, "stage_records") && (value == 0 || value == 1))
        c->stage_records = (int)value;
    else if (!std::strcmp(name, "event_pdl") && (value == 0 || value == 1))
        c->event_pdl = (int)value;
    else if (!std::strcmp(name, "evolve_redraw") && value >= 0 && value <= 2)
        c->evolve_redraw = (int)value;
    else if (!std::strcmp(name, "step_config") && value >= 0 && value <= 1)
        c->step_config = (int)value;
    else if (!std::strcmp(name, "step_spill") && (value == 0 || value == 1))
        c->step_spill = (int)value;
    else if (!std::strcmp(name, "step_batch_wait") && value >= 0 && value <= 64)
        c->step_batch_wait = (int)value;
    else if (!std::strcmp(name, "host_slabs") && value >= 0 && value <= kMaxSlabs)
        c->host_slabs = (int)value;
    else
        return fail(c, PICSARQED_ERR_INVALID, std::string("unknown option or bad value: ") + name);
    return PICSARQED_OK;
}

// PAPER.md:275.  CODATA 2018: c, h, e exact; m_e, alpha recommended values (qed_device.cuh).
int picsarqed_set_units(picsarqed_ctx* c, int system, double reference) {
    if (!c) return PICSARQED_ERR_INVALID;
    constexpr double kCharge = 1.602176634e-19;                       // C
    constexpr double kHbar = kPlanck / (2.0 * kPi);                   // J s
    constexpr double kMc = kElectronMass * kLightSpeed;               // m_e c, kg m/s
    constexpr double kEs = kElectronMass * kElectronMass * kLightSpeed * kLightSpeed * kLightSpeed / (kCharge * kHbar);  // V/m
    constexpr double kMeV = 1e6 * kCharge;                            // J
    constexpr double kMassMeV = kElectronMass * kLightSpeed * kLightSpeed / kMeV;  // m_e c^2 in MeV
    double sp = 1.0, se = 1.0, sb = 1.0, st = 1.0;
    switch (system) {
        case PICSARQED_UNITS_LIBRARY: break;
        case PICSARQED_UNITS_SI:            // kg m/s, V/m, T, s
            sp = 1.0 / kMc;
            se = 1.0 / kEs;
            sb = kLightSpeed / kEs;
            break;
        case PICSARQED_UNITS_NORM_OMEGA:    // c = e = m_e = 1 and a reference angular frequency omega [1/s]:
            if (!(reference > 0.0)) return fail(c, PICSARQED_ERR_INVALID, "set_units: reference frequency must be > 0");
            se = sb = kElectronMass * kLightSpeed * reference / kCharge / kEs;  // E unit m c omega/e, B unit m omega/e
            st = 1.0 / reference;
            break;
        case PICSARQED_UNITS_NORM_LAMBDA:   // the same with a reference length lambda [m]: omega = c/lambda
            if (!(reference > 0.0)) return fail(c, PICSARQED_ERR_INVALID, "set_units: reference length must be > 0");
            se = sb = kElectronMass * kLightSpeed * kLightSpeed / (kCharge * reference) / kEs;
            st = reference / kLightSpeed;
            break;
        case PICSARQED_UNITS_HL_MEV:        // Heaviside-Lorentz natural units (hbar = c = 1), 1 MeV: p in MeV, E and
            sp = 1.0 / kMassMeV;            // B in MeV^2, t in 1/MeV; e_HL = sqrt(4 pi alpha), E_s = m^2/e_HL
            se = sb = std::sqrt(4.0 * kPi * kFineStructure) / (kMassMeV * kMassMeV);
            st = kHbar / kMeV;
            break;
        default: return fail(c, PICSARQED_ERR_INVALID, "set_units: unknown unit system");
    }
    c->units.p = sp;
    c->units.e = se;
    c->units.b = sb;
    c->units.inv_p = 1.0 / sp;
    c->t_scale = st;
    c->unit_system = system;
    return PICSARQED_OK;
}

int picsarqed_get_unit_scales(picsarqed_ctx* c, double* scales) {
    if (!c || !scales) return PICSARQED_ERR_INVALID;
    scales[0] = c->units.p;
    scales[1] = c->units.e;
    scales[2] = c->units.b;
    scales[3] = c->t_scale;
    return PICSARQED_OK;
}

int picsarqed_get_timing(picsarqed_ctx* c, double* host_ms, long long* host_calls) {
    if (!c || !host_ms || !host_calls) return PICSARQED_ERR_INVALID;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    host_ms[0] = host_ms[1] = 0.0;
    *host_calls = (long long)(c->timing_events.size() / 3);
    for (size_t k = 0; k + 2 < c->timing_events.size(); k += 3) {
        float a = 0.f, b = 0.f;
        cudaEventElapsedTime(&a, c->timing_events[k], c->timing_events[k + 1]);
        cudaEventElapsedTime(&b, c->timing_events[k + 1], c->timing_events[k + 2]);
        host_ms[0] += a;
        host_ms[1] += b;
    }
    for (cudaEvent_t e : c->timing_events) cudaEventDestroy(e);
    c->timing_events.clear();
    return PICSARQED_OK;
}

int picsarqed_import_tables(picsarqed_ctx* c, const picsarqed_table_params* p, const double* lnG,
                            const double* qs_lnP, const double* lnT, const double* bw_P) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (!params_ok(p) || !lnG || !qs_lnP || !lnT || !bw_P) return fail(c, PICSARQED_ERR_INVALID, "bad table arguments");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    c->have_tables = false;
    if (int rc = alloc_tables(c, *p)) return rc;
    const double* src[4] = {lnG, qs_lnP, lnT, bw_P};
    for (int k = 0; k < 4; ++k)
        PXQ_CUDA(c, cudaMemcpyAsync(c->tab64[k], src[k], c->tab_n[k] * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    if (int rc = narrow_tables(c)) return rc;
    if (int rc = build_guides(c)) return rc;
    PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_tables = true;
    return PICSARQED_OK;
}

int picsarqed_export_tables(picsarqed_ctx* c, int which, double* host_dst, size_t n_elems) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables");
    if (which < 0 || which > 3 || !host_dst || n_elems != c->tab_n[which])
        return fail(c, PICSARQED_ERR_INVALID, "bad export arguments");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    PXQ_CUDA(c, cudaMemcpyAsync(host_dst, c->tab64[which], n_elems * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    return PICSARQED_OK;
}

int picsarqed_read_count(picsarqed_ctx* c, const unsigned long long* d_count, unsigned long long* host_out) {
    if (!c || !d_count || !host_out) return PICSARQED_ERR_INVALID;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    PXQ_CUDA(c, cudaMemcpyAsync(host_out, d_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    return PICSARQED_OK;
}

}  // extern "C"

// =====================================================================================
//  launchers
// =====================================================================================
namespace {

int stream_grid(const picsarqed_ctx* c, long long work_items, int per_block) {
    const long long blocks = (work_items + per_block - 1) / per_block;
    return (int)std::max<long long>(1, std::min<long long>(blocks, (long long)c->num_sms * 8));
}

template <typename R, int SPECIES>
int launch_chi(picsarqed_ctx* c, long long n, const void* const* a, void* out) {
    constexpr int V = 16 / sizeof(R);
    chi_kernel<R, SPECIES><<<stream_grid(c, (n + V - 1) / V, 256), 256, 0, c->stream>>>(
        (const R*)a[0], (const R*)a[1], (const R*)a[2], (const R*)a[3], (const R*)a[4], (const R*)a[5],
        (const R*)a[6], (const R*)a[7], (const R*)a[8], (R*)out, n, c->units);
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

struct StageView { unsigned char* rec; unsigned short* cnt; unsigned int* tile_sum; int chunks_per_tile; long long stride; int remove_photons;
                   int redraw_tau = 0; unsigned long long seed = 0, step = 0, id_base = 0; };

template <typename R, typename TR, int SPECIES, int U, bool EMIT>
int launch_evolve_u(picsarqed_ctx* c, long long n, const void* const* a, double dt, void* tau,
                    unsigned long long* d_n_events, StageView sv = StageView{nullptr, nullptr, nullptr, 1, 0, 0}) {
    constexpr int V = 16 / sizeof(R);
    constexpr int TILE = kEvolveThreads * V * U;
    EvolveArgs<R, TR> args;
    for (int k = 0; k < 3; ++k) {
        args.p[k] = (const R*)a[k];
        args.e[k] = (const R*)a[3 + k];
        args.b[k] = (const R*)a[6 + k];
    }
    args.tau = (TR*)tau;
    args.n = n;
    args.tab = view_1d<R>(c, SPECIES);
    args.rate_dt = (SPECIES == 0 ? 2.0 / 3.0 : 1.0) * kAlphaOverTauC * (dt * c->t_scale);  // dt in the caller's time unit
    args.units = c->units;
    args.partials = c->partials;
    args.ticket = c->ticket;
    args.d_n_events = d_n_events;
    args.stage_rec = sv.rec;
    args.stage_stride = sv.stride;
    args.stage_cnt = sv.cnt;
    args.tile_sum = sv.tile_sum;
    args.chunks_per_tile = sv.chunks_per_tile;
    args.remove_photons = sv.remove_photons;
    args.redraw_tau = sv.redraw_tau;
    args.seed = sv.seed;
    args.step = sv.step;
    args.id_base = sv.id_base;
    size_t smem = ((size_t)args.tab.n * sizeof(R) + 127) & ~(size_t)127;
    args.table_in_smem = smem <= 96 * 1024;  // larger tables are read through L1/L2
    if (!args.table_in_smem) smem = 0;
    args.table_bytes = (unsigned)smem;
    if (EMIT) smem += (size_t)(kEvolveThreads / 32) * kStageCap * StageRecord<R>::kBytes;
    // (the scaled variant only when the caller's arrays are in another unit system: the default path pays nothing)
    auto kern = c->unit_system != PICSARQED_UNITS_LIBRARY ? evolve_kernel<R, TR, SPECIES, U, EMIT, true>
                                                          : evolve_kernel<R, TR, SPECIES, U, EMIT, false>;
    if (smem > 48 * 1024) PXQ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    PXQ_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kEvolveThreads, smem));
    if (per_sm < 1) per_sm = 1;
    if (c->evolve_ctas_per_sm > 0) per_sm = std::min(per_sm, c->evolve_ctas_per_sm);
    const long long ntiles = (n + TILE - 1) / TILE;
    const int grid = (int)std::max<long long>(1, std::min<long long>(ntiles, (long long)c->num_sms * per_sm));
    if (grid > c->partials_cap) return fail(c, PICSARQED_ERR_CUDA, "internal: partials too small");
    kern<<<grid, kEvolveThreads, smem, c->stream>>>(args);
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

// per-chunk scratch: [tile sums][records][counts][offsets]
struct ChunkScratch { unsigned char* rec; unsigned short* cnt; unsigned long long* off; unsigned int* sum; long long n_chunks; long long stride; };

// seg_bytes: bytes of one entry of a chunk's segment (a staged record, or a staged result of the fused step; 0 = none)
int chunk_scratch(picsarqed_ctx* c, long long n, size_t seg_bytes, ChunkScratch* out, bool keep_staged = false) {
    if (c->staged_valid && !keep_staged) {
        // records staged by evolve_optical_depth were never consumed: their tile sums must not leak into this call
        if (c->rec) PXQ_CUDA(c, cudaMemsetAsync(c->rec, 0, c->rec_sum_bytes, c->stream));
        c->staged_valid = false;
    }
    const long long nchunks = (n + kChunk - 1) / kChunk;
    const size_t rec_sz = ((size_t)nchunks * kStageCap * seg_bytes + 255) & ~(size_t)255;
    const size_t cnt_sz = ((size_t)nchunks * sizeof(unsigned short) + 255) & ~(size_t)255;
    // tiles hold at least 8 chunks: n_chunks/8 + 1 tile offsets and tile sums are always enough
    const size_t off_sz = ((size_t)(nchunks / 8 + 2) * sizeof(unsigned long long) + 255) & ~(size_t)255;
    const size_t sum_sz = ((size_t)(nchunks / 8 + 2) * sizeof(unsigned int) + 255) & ~(size_t)255;
    // the tile sums live at the FRONT of the buffer (their place must not move with n: they are kept at zero
    // between calls), then records, counts, offsets
    const size_t body = rec_sz + cnt_sz + off_sz;
    if (sum_sz > c->rec_sum_bytes || c->rec_sum_bytes + body > c->rec_bytes) {
        // grow (synchronises): half as much again when a population creeps up step after step (closed loop),
        // exact the first time
        PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
        const bool headroom = c->rec_bytes > 0;
        const size_t sum_want = headroom ? (sum_sz + sum_sz / 2 + 255) & ~(size_t)255 : sum_sz;
        const size_t want = sum_want + (headroom ? body + body / 2 : body);
        if (c->rec) cudaFree(c->rec);
        c->rec = nullptr;
        c->rec_bytes = 0;
        c->rec_sum_bytes = 0;
        PXQ_CUDA(c, cudaMalloc(&c->rec, want));
        PXQ_CUDA(c, cudaMemsetAsync(c->rec, 0, sum_want, c->stream));   // tile sums start (and are kept) at zero
        c->rec_bytes = want;
        c->rec_sum_bytes = sum_want;
    }
    out->sum = static_cast<unsigned int*>(c->rec);
    out->rec = static_cast<unsigned char*>(c->rec) + c->rec_sum_bytes;
    out->cnt = reinterpret_cast<unsigned short*>(out->rec + rec_sz);
    out->off = reinterpret_cast<unsigned long long*>(out->rec + rec_sz + cnt_sz);
    out->n_chunks = nchunks;
    out->stride = (long long)(kStageCap * seg_bytes);
    return PICSARQED_OK;
}

// chunks per tile of the configured event_kernel shape
int event_chunks_per_tile(const picsarqed_ctx* c) {
    (void)c;
    return kEventTileChunks;  // both shapes of launch_event_pass (the counting kernels rely on it)
}

template <typename R, typename TR, int SPECIES>
int launch_evolve(picsarqed_ctx* c, long long n, const void* const* a, double dt, void* tau,
                  unsigned long long* d_n_events) {
    if (c->stage_records) {
        // the pass of qed_step without the removal of photons: tau evolves, the records of what fired are staged
        ChunkScratch cs;
        if (int rc = chunk_scratch(c, n, StageRecord<R>::kBytes, &cs)) return rc;
        StageView sv{cs.rec, cs.cnt, cs.sum, event_chunks_per_tile(c), cs.stride, 0};
        constexpr int U = kChunk / (32 * (16 / (int)sizeof(R)));
        if (int rc = launch_evolve_u<R, TR, SPECIES, U, true>(c, n, a, dt, tau, d_n_events, sv)) return rc;
        constexpr long long kTile = (long long)kEvolveThreads * (16 / (int)sizeof(R)) * U;
        if (n % kTile)
            count_chunks_kernel<TR><<<1, 256, 0, c->stream>>>((const TR*)tau, n, (n / kTile) * kTile / kChunk, cs.n_chunks, cs.cnt,
                                                              cs.sum, sv.chunks_per_tile);
        PXQ_CUDA(c, cudaGetLastError());
        c->staged_valid = true;
        c->staged_tau = tau;
        c->staged_n = n;
        c->staged_species = SPECIES;
        c->staged_dtype = sizeof(R) == 8;
        c->staged_tau_dtype = sizeof(TR) == 8;
        return PICSARQED_OK;
    }
    // measured on B200: two 128-bit loads per array per thread, except fp32 photons (branchier: one)
    int u = c->evolve_unroll ? c->evolve_unroll : ((sizeof(R) == 4 && SPECIES == 1) ? 1 : 2);
    if (u == 1) return launch_evolve_u<R, TR, SPECIES, 1, false>(c, n, a, dt, tau, d_n_events);
    if (u == 4) return launch_evolve_u<R, TR, SPECIES, 4, false>(c, n, a, dt, tau, d_n_events);
    return launch_evolve_u<R, TR, SPECIES, 2, false>(c, n, a, dt, tau, d_n_events);
}

// levels 2 and 3 of the compaction: chunk counts (and their tile sums) -> offsets -> events
template <typename R, typename TR, int KIND>
int launch_event_pass(picsarqed_ctx* c, long long n, const ChunkScratch& cs, void* const* p, const void* const* eb,
                      void* tau, unsigned long long seed, unsigned long long step, unsigned long long id_base,
                      long long capacity, void* const* out_p, void* const* out_tau, long long* parent,
                      unsigned long long* d_n_out) {
    EventArgs<R, TR> ev;
    for (int k = 0; k < 3; ++k) {
        ev.p[k] = (R*)p[k];
        ev.e[k] = (const R*)eb[k];
        ev.b[k] = (const R*)eb[3 + k];
    }
    ev.tau = (TR*)tau;
    ev.n = n;
    ev.cdf = view_2d<R>(c, KIND);
    ev.seed = seed;
    ev.step = step;
    ev.id_base = id_base;
    ev.capacity = capacity;
    for (int k = 0; k < 6; ++k) ev.out_p[k] = (R*)out_p[k];
    for (int k = 0; k < 2; ++k) ev.out_tau[k] = (TR*)out_tau[k];
    ev.parent = parent;
    ev.stage_rec = cs.rec;
    ev.stage_stride = cs.stride;
    ev.stage_cnt = cs.cnt;
    ev.tile_offset = cs.off;
    ev.slot_base = c->link_slot_base;
    ev.parent_base = c->link_parent_base;
    ev.units = c->units;
    const int chunks = event_chunks_per_tile(c);
    const long long n_tiles = (cs.n_chunks + chunks - 1) / chunks;
    tile_scan_kernel<<<1, kScanThreads, 0, c->stream>>>(cs.cnt, cs.n_chunks, chunks, n_tiles, cs.off, c->link_slot_base, d_n_out,
                                                        nullptr, cs.sum);
#define PXQ_LAUNCH_EVENTS(T, CH, MB)                                                                         \
    do {                                                                                                     \
        auto kern = event_kernel<R, TR, KIND, T, CH, MB>;                                                    \
        int per_sm = 0;                                                                                      \
        PXQ_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T, 0));                     \
        const unsigned grid = (unsigned)std::max<long long>(                                                 \
            1, std::min<long long>(n_tiles, (long long)c->num_sms * std::max(per_sm, 1)));                   \
        /* programmatic dependent launch: the CTAs become resident while the offsets scan (one CTA) still runs and wait   \
           for it at griddepcontrol.wait -- the launch latency of this kernel is off the step's critical path */        \
        cudaLaunchConfig_t cfg{};                                                                            \
        cfg.gridDim = dim3(grid);                                                                            \
        cfg.blockDim = dim3(T);                                                                              \
        cfg.stream = c->stream;                                                                              \
        cudaLaunchAttribute at[1];                                                                           \
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                                       \
        at[0].val.programmaticStreamSerializationAllowed = c->event_pdl ? 1 : 0;                             \
        cfg.attrs = at;                                                                                      \
        cfg.numAttrs = 1;                                                                                    \
        PXQ_CUDA(c, cudaLaunchKernelEx(&cfg, kern, ev));                                                     \
    } while (0)
    switch (c->event_config) {
        case 1: PXQ_LAUNCH_EVENTS(256, kEventTileChunks, 3); break;
        default: PXQ_LAUNCH_EVENTS(384, kEventTileChunks, 2); break;  // measured best on B200 (config 2: 1-4 us ahead of (256, 24, 3))
    }
#undef PXQ_LAUNCH_EVENTS
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

// generate_photons / generate_pairs: count the chunks from tau, then the common event pass
template <typename R, typename TR, int KIND>
int launch_events(picsarqed_ctx* c, long long n, void* const* p, const void* const* eb, void* tau,
                  unsigned long long seed, unsigned long long step, unsigned long long id_base, long long capacity,
                  void* const* out_p, void* const* out_tau, long long* parent, unsigned long long* d_n_out) {
    ChunkScratch cs;
    if (c->staged_valid && c->staged_tau == tau && c->staged_n == n && c->staged_species == KIND &&
        c->staged_dtype == (int)(sizeof(R) == 8) && c->staged_tau_dtype == (int)(sizeof(TR) == 8)) {
        // "stage_records": the evolve call before this one staged the records and counted the chunks
        if (int rc = chunk_scratch(c, n, StageRecord<R>::kBytes, &cs, true)) return rc;
        c->staged_valid = false;
        return launch_event_pass<R, TR, KIND>(c, n, cs, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau, parent,
                                              d_n_out);
    }
    if (int rc = chunk_scratch(c, n, 0, &cs)) return rc;
    const int grid = (int)std::max<long long>(1, std::min<long long>((cs.n_chunks + 7) / 8, (long long)c->num_sms * 8));
    count_chunks_kernel<TR><<<grid, 256, 0, c->stream>>>((const TR*)tau, n, 0, cs.n_chunks, cs.cnt, cs.sum,
                                                         event_chunks_per_tile(c));
    return launch_event_pass<R, TR, KIND>(c, n, cs, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau, parent,
                                          d_n_out);
}

// the unstaged path of launch_events on a scratch the caller laid out (picsarqed_generate_photons_noalloc: the static array)
template <typename R, typename TR, int KIND>
int launch_events_on(picsarqed_ctx* c, long long n, const ChunkScratch& cs, void* const* p, const void* const* eb, void* tau,
                     unsigned long long seed, unsigned long long step, unsigned long long id_base, long long capacity,
                     void* const* out_p, void* const* out_tau, long long* parent, unsigned long long* d_n_out) {
    const int grid = (int)std::max<long long>(1, std::min<long long>((cs.n_chunks + 7) / 8, (long long)c->num_sms * 8));
    count_chunks_kernel<TR><<<grid, 256, 0, c->stream>>>((const TR*)tau, n, 0, cs.n_chunks, cs.cnt, cs.sum,
                                                         event_chunks_per_tile(c));
    return launch_event_pass<R, TR, KIND>(c, n, cs, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau, parent,
                                          d_n_out);
}

// the three timing events of a step ("time_kernels"): handed to the context when the step was enqueued, destroyed otherwise
struct StepEvents {
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    bool kept = false;
    ~StepEvents() {
        if (!kept)
            for (cudaEvent_t e : ev)
                if (e) cudaEventDestroy(e);
    }
};

// qed_step, fused (step.cuh): streaming warps evolve, event warps of the same CTA generate the events and rewrite the
// parents while their sectors are in L2; then the offsets scan and the placement of the staged secondaries
template <typename R, typename TR, int SPECIES, int EW, int D, int REG_S, int REG_E>
int launch_fused_step_c(picsarqed_ctx* c, long long n, void* const* p, const void* const* eb, void* tau, double dt,
                        unsigned long long seed, unsigned long long step, unsigned long long id_base, long long capacity,
                        void* const* out_p, void* const* out_tau, long long* parent, unsigned long long* d_n_out) {
    constexpr int SW = 16, NS = 2;
    typedef StepLayout<R, TR, SW, EW, D, NS> L;
    constexpr int THREADS = L::THREADS;
    constexpr long long kTile = (long long)SW * kChunk;
    typedef StepResult<R, TR, SPECIES> Res;
    ChunkScratch cs;
    if (int rc = chunk_scratch(c, n, std::max<size_t>(sizeof(Res), StageRecord<R>::kBytes), &cs)) return rc;
    StepArgs<R, TR, SPECIES> sa;
    EvolveArgs<R, TR>& args = sa.ev;
    for (int k = 0; k < 3; ++k) {
        args.p[k] = (const R*)p[k];
        args.e[k] = (const R*)eb[k];
        args.b[k] = (const R*)eb[3 + k];
        sa.ge.p[k] = (R*)p[k];
        sa.ge.e[k] = (const R*)eb[k];
        sa.ge.b[k] = (const R*)eb[3 + k];
    }
    args.tau = (TR*)tau;
    args.n = n;
    args.tab = view_1d<R>(c, SPECIES);
    args.rate_dt = (SPECIES == 0 ? 2.0 / 3.0 : 1.0) * kAlphaOverTauC * (dt * c->t_scale);
    args.units = c->units;
    args.partials = nullptr;
    args.ticket = nullptr;
    args.d_n_events = nullptr;
    args.stage_rec = nullptr;
    args.stage_stride = cs.stride;
    args.stage_cnt = cs.cnt;
    args.tile_sum = cs.sum;
    args.chunks_per_tile = event_chunks_per_tile(c);
    args.remove_photons = 0;
    args.redraw_tau = 0;
    args.seed = args.step = args.id_base = 0;
    // shared memory: [1D table][sub-chunk stages][record queues]; a table that does not fit beside them is read through L1
    constexpr size_t kSmemMax = 227 * 1024 - 2048;   // (2 KB: the kernel's static shared memory)
    size_t smem = ((size_t)args.tab.n * sizeof(R) + 127) & ~(size_t)127;
    args.table_in_smem = smem + L::stages_bytes + L::queue_bytes <= kSmemMax;
    if (!args.table_in_smem) smem = 0;
    args.table_bytes = (unsigned)smem;
    smem += L::stages_bytes + L::queue_bytes;
    sa.ge.tau = (TR*)tau;
    sa.ge.n = n;
    sa.ge.cdf = view_2d<R>(c, SPECIES);
    sa.ge.seed = seed;
    sa.ge.step = step;
    sa.ge.id_base = id_base;
    sa.ge.capacity = capacity;
    for (int k = 0; k < 6; ++k) sa.ge.out_p[k] = nullptr;
    for (int k = 0; k < 2; ++k) sa.ge.out_tau[k] = nullptr;
    sa.ge.parent = nullptr;
    sa.ge.stage_rec = nullptr;
    sa.ge.stage_stride = cs.stride;
    sa.ge.stage_cnt = nullptr;
    sa.ge.tile_offset = nullptr;
    sa.ge.slot_base = nullptr;
    sa.ge.parent_base = 0;
    sa.ge.units = c->units;
    sa.stage_res = cs.rec;
    sa.spill = c->step_spill;
    sa.batch_wait = c->step_batch_wait;
    const bool scaled = c->unit_system != PICSARQED_UNITS_LIBRARY;
    // registers (REG_S, REG_E != 0): the launch gives every thread floor(64 Ki / THREADS) rounded down to a multiple of 8
    // (72 for 896 threads); the streaming warps hand some back and the event warps take them
    void (*kern)(StepArgs<R, TR, SPECIES>) =
        scaled ? step_kernel<R, TR, SPECIES, true, SW, EW, D, NS, REG_S, REG_E> : step_kernel<R, TR, SPECIES, false, SW, EW, D, NS, REG_S, REG_E>;
    if (REG_S != 0) {
        cudaFuncAttributes fa;
        PXQ_CUDA(c, cudaFuncGetAttributes(&fa, kern));
        if ((long long)fa.numRegs * THREADS < (long long)SW * 32 * REG_S + (long long)(THREADS - SW * 32) * REG_E)
            return fail(c, PICSARQED_ERR_CUDA, "internal: the fused step kernel was built with too few registers for setmaxnreg");
    }
    PXQ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const long long ntiles = n / kTile;
    const int grid = (int)std::max<long long>(1, std::min<long long>(ntiles, (long long)c->num_sms));
    StepEvents se;
    cudaEvent_t* ev = se.ev;
    if (c->time_kernels) {
        for (int k = 0; k < 3; ++k) PXQ_CUDA(c, cudaEventCreate(&ev[k]));
        PXQ_CUDA(c, cudaEventRecord(ev[0], c->stream));
    }
    kern<<<grid, THREADS, smem, c->stream>>>(sa);
    PXQ_CUDA(c, cudaGetLastError());
    if (n % kTile)  // the ragged last tile stages nothing: count its chunks from the updated tau
        count_chunks_kernel<TR><<<1, 256, 0, c->stream>>>((const TR*)tau, n, (n / kTile) * kTile / kChunk, cs.n_chunks, cs.cnt,
                                                          cs.sum, args.chunks_per_tile);
    if (c->time_kernels) PXQ_CUDA(c, cudaEventRecord(ev[1], c->stream));
    if (int rc = launch_event_pass<R, TR, SPECIES>(c, n, cs, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau,
                                                   parent, d_n_out))
        return rc;
    if (c->time_kernels) {
        PXQ_CUDA(c, cudaEventRecord(ev[2], c->stream));
        for (int k = 0; k < 3; ++k) c->timing_events.push_back(ev[k]);
        se.kept = true;
    }
    return PICSARQED_OK;
}

template <typename R, typename TR, int SPECIES>
int launch_fused_step(picsarqed_ctx* c, long long n, void* const* p, const void* const* eb, void* tau, double dt,
                      unsigned long long seed, unsigned long long step, unsigned long long id_base, long long capacity,
                      void* const* out_p, void* const* out_tau, long long* parent, unsigned long long* d_n_out) {
    // "step_config": 0 = 16 streaming warps in 80 registers + 12 event warps in 56; 1 = 16 + 8 event warps, all in 80
#define PXQ_FUSED(EW, D, RS, RE)                                                                                         \
    return launch_fused_step_c<R, TR, SPECIES, EW, D, RS, RE>(c, n, p, eb, tau, dt, seed, step, id_base, capacity, out_p, \
                                                              out_tau, parent, d_n_out)
    if (c->step_config == 1) PXQ_FUSED(8, 3, 0, 0);
    PXQ_FUSED(12, 3, 80, 56);
#undef PXQ_FUSED
}

// qed_step: the evolve pass stages the records of the particles that fire, then the common event pass
template <typename R, typename TR, int SPECIES>
int launch_step(picsarqed_ctx* c, long long n, void* const* p, const void* const* eb, void* tau, double dt,
                unsigned long long seed, unsigned long long step, unsigned long long id_base, long long capacity,
                void* const* out_p, void* const* out_tau, long long* parent, unsigned long long* d_n_out) {
    if (c->fused_step)
        return launch_fused_step<R, TR, SPECIES>(c, n, p, eb, tau, dt, seed, step, id_base, capacity, out_p, out_tau, parent,
                                                 d_n_out);
    ChunkScratch cs;
    if (int rc = chunk_scratch(c, n, StageRecord<R>::kBytes, &cs)) return rc;
    StageView sv;
    sv.rec = cs.rec;
    sv.stride = cs.stride;
    sv.cnt = cs.cnt;
    sv.tile_sum = cs.sum;
    sv.chunks_per_tile = event_chunks_per_tile(c);
    sv.remove_photons = 1;
    // "evolve_redraw": 0 = the event pass re-draws the parents' optical depth, 1 = the evolve pass does, for fp64 particles
    // (whose evolve pass waits for HBM and has the issue slots), 2 = for every dtype
    sv.redraw_tau = SPECIES == 0 && (c->evolve_redraw == 2 || (c->evolve_redraw == 1 && sizeof(R) == 8)) ? 1 : 0;
    sv.seed = seed;
    sv.step = step;
    sv.id_base = id_base;
    const void* a9[9] = {p[0], p[1], p[2], eb[0], eb[1], eb[2], eb[3], eb[4], eb[5]};
    constexpr int U = kChunk / (32 * (16 / (int)sizeof(R)));  // fp64: 2, fp32: 1
    StepEvents se;
    cudaEvent_t* ev = se.ev;
    if (c->time_kernels) {
        for (int k = 0; k < 3; ++k) PXQ_CUDA(c, cudaEventCreate(&ev[k]));
        PXQ_CUDA(c, cudaEventRecord(ev[0], c->stream));
    }
    if (int rc = launch_evolve_u<R, TR, SPECIES, U, true>(c, n, a9, dt, tau, nullptr, sv)) return rc;
    constexpr long long kTile = (long long)kEvolveThreads * (16 / (int)sizeof(R)) * U;
    if (n % kTile)  // the ragged last tile stages no records: count its chunks from the updated tau
        count_chunks_kernel<TR><<<1, 256, 0, c->stream>>>((const TR*)tau, n, (n / kTile) * kTile / kChunk, cs.n_chunks, cs.cnt,
                                                          cs.sum, sv.chunks_per_tile);
    if (c->time_kernels) PXQ_CUDA(c, cudaEventRecord(ev[1], c->stream));
    if (int rc = launch_event_pass<R, TR, SPECIES>(c, n, cs, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau,
                                                   parent, d_n_out))
        return rc;
    if (c->time_kernels) {
        PXQ_CUDA(c, cudaEventRecord(ev[2], c->stream));
        for (int k = 0; k < 3; ++k) c->timing_events.push_back(ev[k]);
        se.kept = true;
    }
    return PICSARQED_OK;
}

// dispatch on (dtype, tau_dtype); fp64 particles with fp32 optical depth is not offered
#define PXQ_DISPATCH_RT(ctx, dtype, tau_dtype, CALL)                                       \
    do {                                                                                   \
        if ((dtype) == PICSARQED_F64 && (tau_dtype) == PICSARQED_F64) { typedef double R; typedef double TR; CALL; } \
        else if ((dtype) == PICSARQED_F32 && (tau_dtype) == PICSARQED_F32) { typedef float R; typedef float TR; CALL; } \
        else if ((dtype) == PICSARQED_F32 && (tau_dtype) == PICSARQED_F64) { typedef float R; typedef double TR; CALL; } \
        else return fail(ctx, PICSARQED_ERR_DTYPE, "unsupported (dtype, tau_dtype) combination");                \
    } while (0)

// ordered, filtering append: per-chunk keep counts -> tile offsets -> scatter (cascade.cuh).  d_dst_n (device) overrides
// dst_n when not NULL: the second append of a step starts where the first one ended.
template <typename R, typename TR>
int launch_append(picsarqed_ctx* c, long long m_max, const void* const* s_p, const void* s_tau,
                  const unsigned long long* d_count, double min_energy, void* const* d_p, void* d_tau, long long dst_n,
                  const unsigned long long* d_dst_n, long long dst_capacity, unsigned long long* d_kept,
                  unsigned long long* d_new_n) {
    ChunkScratch cs;
    if (int rc = chunk_scratch(c, m_max, 0, &cs)) return rc;
    const int grid = (int)std::max<long long>(1, std::min<long long>((cs.n_chunks + 7) / 8, (long long)c->num_sms * 8));
    keep_count_kernel<R><<<grid, 256, 0, c->stream>>>((const R*)s_p[0], (const R*)s_p[1], (const R*)s_p[2], d_count, m_max,
                                                       min_energy, cs.n_chunks, cs.cnt);
    const long long n_tiles = (cs.n_chunks + kAppendChunksPerTile - 1) / kAppendChunksPerTile;
    tile_scan_kernel<<<1, kScanThreads, 0, c->stream>>>(cs.cnt, cs.n_chunks, kAppendChunksPerTile, n_tiles, cs.off, nullptr,
                                                        d_kept, d_count, nullptr);
    AppendArgs<R, TR> a;
    for (int k = 0; k < 3; ++k) {
        a.s_p[k] = (const R*)s_p[k];
        a.d_p[k] = (R*)d_p[k];
    }
    a.s_tau = (const TR*)s_tau;
    a.d_tau = (TR*)d_tau;
    a.d_count = d_count;
    a.m_max = m_max;
    a.dst_n = dst_n;
    a.d_dst_n = d_dst_n;
    a.dst_capacity = dst_capacity;
    a.n_chunks = cs.n_chunks;
    a.min_energy = min_energy;
    a.cnt = cs.cnt;
    a.tile_offset = cs.off;
    a.d_kept = d_kept;
    a.d_new_n = d_new_n;
    append_kernel<R, TR><<<grid, 256, 0, c->stream>>>(a);
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

int check_arrays(picsarqed_ctx* c, const void* const* a, int count) {
    for (int k = 0; k < count; ++k)
        if (!a[k] || !aligned16(a[k])) return fail(c, PICSARQED_ERR_INVALID, "null or misaligned array pointer");
    return PICSARQED_OK;
}

}  // namespace

extern "C" {

int picsarqed_chi(picsarqed_ctx* c, int species, int dtype, long long n, const void* px, const void* py,
                  const void* pz, const void* ex, const void* ey, const void* ez, const void* bx, const void* by,
                  const void* bz, void* chi_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || (species != 0 && species != 1)) return fail(c, PICSARQED_ERR_INVALID, "bad n or species");
    if (n == 0) return PICSARQED_OK;
    const void* a[10] = {px, py, pz, ex, ey, ez, bx, by, bz, chi_out};
    if (int rc = check_arrays(c, a, 10)) return rc;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    if (dtype == PICSARQED_F64)
        return species == 0 ? launch_chi<double, 0>(c, n, a, chi_out) : launch_chi<double, 1>(c, n, a, chi_out);
    if (dtype == PICSARQED_F32)
        return species == 0 ? launch_chi<float, 0>(c, n, a, chi_out) : launch_chi<float, 1>(c, n, a, chi_out);
    return fail(c, PICSARQED_ERR_DTYPE, "bad dtype");
}

int picsarqed_schwinger_rate(picsarqed_ctx* c, int dtype, long long n, const void* ex, const void* ey, const void* ez,
                             const void* bx, const void* by, const void* bz, double* rate_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0) return fail(c, PICSARQED_ERR_INVALID, "bad n");
    if (n == 0) return PICSARQED_OK;
    const void* a[7] = {ex, ey, ez, bx, by, bz, rate_out};
    if (int rc = check_arrays(c, a, 7)) return rc;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    if (dtype == PICSARQED_F64)
        schwinger_kernel<double><<<stream_grid(c, (n + 1) / 2, 256), 256, 0, c->stream>>>(
            (const double*)ex, (const double*)ey, (const double*)ez, (const double*)bx, (const double*)by,
            (const double*)bz, rate_out, n, c->units);
    else if (dtype == PICSARQED_F32)
        schwinger_kernel<float><<<stream_grid(c, (n + 3) / 4, 256), 256, 0, c->stream>>>(
            (const float*)ex, (const float*)ey, (const float*)ez, (const float*)bx, (const float*)by, (const float*)bz,
            rate_out, n, c->units);
    else
        return fail(c, PICSARQED_ERR_DTYPE, "bad dtype");
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

int picsarqed_init_optical_depth(picsarqed_ctx* c, int species, int tau_dtype, long long n, unsigned long long seed,
                                 unsigned long long id_base, void* tau) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || (species != 0 && species != 1)) return fail(c, PICSARQED_ERR_INVALID, "bad n or species");
    if (n == 0) return PICSARQED_OK;
    if (!tau || !aligned16(tau)) return fail(c, PICSARQED_ERR_INVALID, "null or misaligned tau");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    const int grid = stream_grid(c, n, 256);
    if (tau_dtype == PICSARQED_F64)
        init_tau_kernel<double><<<grid, 256, 0, c->stream>>>((double*)tau, n, seed, id_base, species);
    else if (tau_dtype == PICSARQED_F32)
        init_tau_kernel<float><<<grid, 256, 0, c->stream>>>((float*)tau, n, seed, id_base, species);
    else
        return fail(c, PICSARQED_ERR_DTYPE, "bad tau_dtype");
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

int picsarqed_evolve_optical_depth(picsarqed_ctx* c, int species, int dtype, int tau_dtype, long long n,
                                   const void* px, const void* py, const void* pz, const void* ex, const void* ey,
                                   const void* ez, const void* bx, const void* by, const void* bz, double dt,
                                   void* tau, unsigned long long* d_n_events) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || (species != 0 && species != 1)) return fail(c, PICSARQED_ERR_INVALID, "bad n or species");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    if (n == 0) {
        if (d_n_events) PXQ_CUDA(c, cudaMemsetAsync(d_n_events, 0, sizeof(unsigned long long), c->stream));
        return PICSARQED_OK;
    }
    const void* a[10] = {px, py, pz, ex, ey, ez, bx, by, bz, tau};
    if (int rc = check_arrays(c, a, 10)) return rc;
    PXQ_DISPATCH_RT(c, dtype, tau_dtype,
                    return species == 0 ? (launch_evolve<R, TR, 0>(c, n, a, dt, tau, d_n_events))
                                        : (launch_evolve<R, TR, 1>(c, n, a, dt, tau, d_n_events)));
}

int picsarqed_generate_photons(picsarqed_ctx* c, int dtype, int tau_dtype, long long n, void* px, void* py, void* pz,
                               const void* ex, const void* ey, const void* ez, const void* bx, const void* by,
                               const void* bz, void* tau, unsigned long long seed, unsigned long long step,
                               unsigned long long id_base, long long capacity, void* ph_px, void* ph_py,
                               void* ph_pz, void* ph_tau, long long* ph_parent, unsigned long long* d_n_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || capacity < 0 || !d_n_out) return fail(c, PICSARQED_ERR_INVALID, "bad n, capacity or d_n_out");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    if (n == 0) {
        PXQ_CUDA(c, cudaMemsetAsync(d_n_out, 0, sizeof(unsigned long long), c->stream));
        return PICSARQED_OK;
    }
    void* p[3] = {px, py, pz};
    const void* eb[6] = {ex, ey, ez, bx, by, bz};
    const void* chk[10] = {px, py, pz, ex, ey, ez, bx, by, bz, tau};
    if (int rc = check_arrays(c, chk, 10)) return rc;
    void* out_p[6] = {ph_px, ph_py, ph_pz, nullptr, nullptr, nullptr};
    void* out_tau[2] = {ph_tau, nullptr};
    if (capacity > 0) {
        const void* o[4] = {ph_px, ph_py, ph_pz, ph_tau};
        if (int rc = check_arrays(c, o, 4)) return rc;
    }
    PXQ_DISPATCH_RT(c, dtype, tau_dtype,
                    return (launch_events<R, TR, 0>(c, n, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau,
                                                    ph_parent, d_n_out)));
}

int picsarqed_generate_pairs(picsarqed_ctx* c, int dtype, int tau_dtype, long long n, void* px, void* py, void* pz,
                             const void* ex, const void* ey, const void* ez, const void* bx, const void* by,
                             const void* bz, void* tau, unsigned long long seed, unsigned long long step,
                             unsigned long long id_base, long long capacity, void* el_px, void* el_py, void* el_pz,
                             void* el_tau, void* po_px, void* po_py, void* po_pz, void* po_tau, long long* parent,
                             unsigned long long* d_n_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || capacity < 0 || !d_n_out) return fail(c, PICSARQED_ERR_INVALID, "bad n, capacity or d_n_out");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    if (n == 0) {
        PXQ_CUDA(c, cudaMemsetAsync(d_n_out, 0, sizeof(unsigned long long), c->stream));
        return PICSARQED_OK;
    }
    void* p[3] = {px, py, pz};
    const void* eb[6] = {ex, ey, ez, bx, by, bz};
    const void* chk[10] = {px, py, pz, ex, ey, ez, bx, by, bz, tau};
    if (int rc = check_arrays(c, chk, 10)) return rc;
    void* out_p[6] = {el_px, el_py, el_pz, po_px, po_py, po_pz};
    void* out_tau[2] = {el_tau, po_tau};
    if (capacity > 0) {
        const void* o[8] = {el_px, el_py, el_pz, el_tau, po_px, po_py, po_pz, po_tau};
        if (int rc = check_arrays(c, o, 8)) return rc;
    }
    PXQ_DISPATCH_RT(c, dtype, tau_dtype,
                    return (launch_events<R, TR, 1>(c, n, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau,
                                                    parent, d_n_out)));
}

// generate_photons on the static scratch: no cudaMalloc, cudaFree or allocating library call on this path
int picsarqed_generate_photons_noalloc(picsarqed_ctx* c, int dtype, int tau_dtype, long long n, void* px, void* py,
                                       void* pz, const void* ex, const void* ey, const void* ez, const void* bx,
                                       const void* by, const void* bz, void* tau, unsigned long long seed,
                                       unsigned long long step, unsigned long long id_base, long long capacity,
                                       void* ph_px, void* ph_py, void* ph_pz, void* ph_tau, long long* ph_parent,
                                       unsigned long long* d_n_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || capacity < 0 || !d_n_out) return fail(c, PICSARQED_ERR_INVALID, "bad n, capacity or d_n_out");
    if (n > kNoAllocMaxN)
        return fail(c, PICSARQED_ERR_INVALID,
                    "generate_photons_noalloc: n = " + std::to_string(n) + " exceeds the static scratch (at most " +
                        std::to_string(kNoAllocMaxN) + " particles per call); use picsarqed_generate_photons");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    void* scratch = nullptr;
    PXQ_CUDA(c, noalloc_scratch_address(c->device, &scratch));
    if (n == 0) {
        PXQ_CUDA(c, cudaMemsetAsync(d_n_out, 0, sizeof(unsigned long long), c->stream));
        return PICSARQED_OK;
    }
    void* p[3] = {px, py, pz};
    const void* eb[6] = {ex, ey, ez, bx, by, bz};
    const void* chk[10] = {px, py, pz, ex, ey, ez, bx, by, bz, tau};
    if (int rc = check_arrays(c, chk, 10)) return rc;
    void* out_p[6] = {ph_px, ph_py, ph_pz, nullptr, nullptr, nullptr};
    void* out_tau[2] = {ph_tau, nullptr};
    if (capacity > 0) {
        const void* o[4] = {ph_px, ph_py, ph_pz, ph_tau};
        if (int rc = check_arrays(c, o, 4)) return rc;
    }
    if (c->staged_valid) {
        // records staged by evolve_optical_depth ("stage_records") describe arrays this call is about to rewrite: dropped
        if (c->rec) PXQ_CUDA(c, cudaMemsetAsync(c->rec, 0, c->rec_sum_bytes, c->stream));
        c->staged_valid = false;
    }
    // [tile sums][counts][offsets]; every call shares the array and finds the last call's contents in it: the tile
    // sums are accumulated by atomics and must start at zero (the counts and offsets are written before they are read)
    ChunkScratch cs;
    cs.sum = static_cast<unsigned int*>(scratch);
    cs.rec = static_cast<unsigned char*>(scratch) + kNoAllocSumBytes;   // no staged records: never dereferenced
    cs.cnt = reinterpret_cast<unsigned short*>(static_cast<unsigned char*>(scratch) + kNoAllocSumBytes);
    cs.off = reinterpret_cast<unsigned long long*>(static_cast<unsigned char*>(scratch) + kNoAllocSumBytes + kNoAllocCntBytes);
    cs.n_chunks = (n + kChunk - 1) / kChunk;
    cs.stride = 0;
    PXQ_CUDA(c, cudaMemsetAsync(cs.sum, 0, kNoAllocSumBytes, c->stream));
    PXQ_DISPATCH_RT(c, dtype, tau_dtype,
                    return (launch_events_on<R, TR, 0>(c, n, cs, p, eb, tau, seed, step, id_base, capacity, out_p, out_tau,
                                                       ph_parent, d_n_out)));
}

}  // extern "C"

extern "C" int picsarqed_qed_step(picsarqed_ctx* c, int species, int dtype, int tau_dtype, long long n, void* px,
                                  void* py, void* pz, const void* ex, const void* ey, const void* ez, const void* bx,
                                  const void* by, const void* bz, void* tau, double dt, unsigned long long seed,
                                  unsigned long long step, unsigned long long id_base, long long capacity,
                                  void* s1_px, void* s1_py, void* s1_pz, void* s1_tau, void* s2_px, void* s2_py,
                                  void* s2_pz, void* s2_tau, long long* parent, unsigned long long* d_n_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || capacity < 0 || !d_n_out || (species != 0 && species != 1))
        return fail(c, PICSARQED_ERR_INVALID, "bad n, capacity, species or d_n_out");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    if (n == 0) {
        PXQ_CUDA(c, cudaMemsetAsync(d_n_out, 0, sizeof(unsigned long long), c->stream));
        return PICSARQED_OK;
    }
    void* p[3] = {px, py, pz};
    const void* eb[6] = {ex, ey, ez, bx, by, bz};
    const void* chk[10] = {px, py, pz, ex, ey, ez, bx, by, bz, tau};
    if (int rc = check_arrays(c, chk, 10)) return rc;
    void* out_p[6] = {s1_px, s1_py, s1_pz, s2_px, s2_py, s2_pz};
    void* out_tau[2] = {s1_tau, s2_tau};
    if (capacity > 0) {
        const void* o[8] = {s1_px, s1_py, s1_pz, s1_tau, s2_px, s2_py, s2_pz, s2_tau};
        if (int rc = check_arrays(c, o, species == 0 ? 4 : 8)) return rc;
    }
    PXQ_DISPATCH_RT(c, dtype, tau_dtype,
                    return species == 0 ? (launch_step<R, TR, 0>(c, n, p, eb, tau, dt, seed, step, id_base, capacity,
                                                                 out_p, out_tau, parent, d_n_out))
                                        : (launch_step<R, TR, 1>(c, n, p, eb, tau, dt, seed, step, id_base, capacity,
                                                                 out_p, out_tau, parent, d_n_out)));
}

// =====================================================================================
//  host-buffer path (end-to-end timing): H2D copies, evolve + events, D2H copies
// =====================================================================================
extern "C" int picsarqed_step_host(picsarqed_ctx* c, int species, int dtype, int tau_dtype, long long n, void* h_px,
                                   void* h_py, void* h_pz, const void* h_ex, const void* h_ey, const void* h_ez,
                                   const void* h_bx, const void* h_by, const void* h_bz, void* h_tau, double dt,
                                   unsigned long long seed, unsigned long long step, unsigned long long id_base,
                                   long long capacity, void* const* h_sec, long long* h_parent,
                                   unsigned long long* h_n_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || capacity < 0 || !h_n_out || (species != 0 && species != 1))
        return fail(c, PICSARQED_ERR_INVALID, "bad n, capacity, species or h_n_out");
    if ((dtype != 0 && dtype != 1) || (tau_dtype != 0 && tau_dtype != 1) || (dtype == 1 && tau_dtype == 0))
        return fail(c, PICSARQED_ERR_DTYPE, "unsupported (dtype, tau_dtype) combination");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    *h_n_out = 0;
    if (n == 0) return PICSARQED_OK;
    const size_t es = dtype ? 8 : 4, ts = tau_dtype ? 8 : 4;
    auto pad = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const int n_sec = species == 0 ? 3 : 6, n_sec_tau = species == 0 ? 1 : 2;
    const size_t a_bytes = pad((size_t)n * es), t_bytes = pad((size_t)n * ts);
    const size_t sp_bytes = pad((size_t)capacity * es), st_bytes = pad((size_t)capacity * ts);
    const size_t par_bytes = pad((size_t)capacity * sizeof(long long));
    const size_t need = 9 * a_bytes + t_bytes + n_sec * sp_bytes + n_sec_tau * st_bytes + par_bytes;
    if (need > c->stage_bytes) {
        PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
        if (c->stage) cudaFree(c->stage);
        c->stage = nullptr;
        c->stage_bytes = 0;
        PXQ_CUDA(c, cudaMalloc(&c->stage, need));
        c->stage_bytes = need;
    }
    char* base = static_cast<char*>(c->stage);
    void* d[10];
    for (int k = 0; k < 9; ++k) d[k] = base + k * a_bytes;
    d[9] = base + 9 * a_bytes;
    char* sec0 = base + 9 * a_bytes + t_bytes;
    void* d_sec_p[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    void* d_sec_tau[2] = {nullptr, nullptr};
    for (int k = 0; k < n_sec; ++k) d_sec_p[k] = sec0 + k * sp_bytes;
    for (int k = 0; k < n_sec_tau; ++k) d_sec_tau[k] = sec0 + n_sec * sp_bytes + k * st_bytes;
    long long* d_parent = reinterpret_cast<long long*>(sec0 + n_sec * sp_bytes + n_sec_tau * st_bytes);

    const void* h_in[10] = {h_px, h_py, h_pz, h_ex, h_ey, h_ez, h_bx, h_by, h_bz, h_tau};
    for (int k = 0; k < 10; ++k)
        if (!h_in[k]) return fail(c, PICSARQED_ERR_INVALID, "null host array");
    void* h_back[4] = {h_px, h_py, h_pz, h_tau};
    const int back_of[4] = {0, 1, 2, 9};

    // Slabs of whole evolve tiles, at least 1 Mi particles each: while slab k is stepped, slab k+1 is on its way
    // in and slab k-1 on its way out (PCIe is full duplex; the copies are asynchronous for pinned host memory).
    // The slabs are stepped in order on one stream and chained through d_counts, so the results (secondaries,
    // their order, the capacity rule) are those of one qed_step over the whole array.
    long long slab = n;
    int n_slabs = 1;
    {
        const long long kMinSlab = 1 << 20;
        int want = c->host_slabs > 0 ? c->host_slabs : (int)std::min<long long>(32, n / kMinSlab);
        if (want > 1) {
            slab = ((n + want - 1) / want + 1023) / 1024 * 1024;
            n_slabs = (int)((n + slab - 1) / slab);
        }
    }
    if (!c->h2d_stream) PXQ_CUDA(c, cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking));
    if (!c->d2h_stream) PXQ_CUDA(c, cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking));
    while ((int)c->slab_events.size() < 2 * n_slabs) {
        cudaEvent_t e;
        PXQ_CUDA(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        c->slab_events.push_back(e);
    }
    struct LinkReset {  // the link must not outlive this call, whatever path leaves it -- and no copy into or out of the
        picsarqed_ctx* c;   // caller's host buffers may still be in flight when the call returns, error or not
        ~LinkReset() {
            c->link_slot_base = nullptr;
            c->link_parent_base = 0;
            cudaStreamSynchronize(c->h2d_stream);
            cudaStreamSynchronize(c->stream);
            cudaStreamSynchronize(c->d2h_stream);
        }
    } link_reset{c};
    PXQ_CUDA(c, cudaMemsetAsync(c->d_counts, 0, sizeof(unsigned long long), c->stream));
    for (int s = 0; s < n_slabs; ++s) {
        const long long i0 = (long long)s * slab, m = std::min(slab, n - i0);
        cudaEvent_t copied_in = c->slab_events[2 * s], stepped = c->slab_events[2 * s + 1];
        for (int k = 0; k < 10; ++k) {
            const size_t w = k == 9 ? ts : es;
            PXQ_CUDA(c, cudaMemcpyAsync(static_cast<char*>(d[k]) + (size_t)i0 * w,
                                        static_cast<const char*>(h_in[k]) + (size_t)i0 * w, (size_t)m * w,
                                        cudaMemcpyHostToDevice, c->h2d_stream));
        }
        PXQ_CUDA(c, cudaEventRecord(copied_in, c->h2d_stream));
        PXQ_CUDA(c, cudaStreamWaitEvent(c->stream, copied_in, 0));
        void* ds[10];
        for (int k = 0; k < 10; ++k) ds[k] = static_cast<char*>(d[k]) + (size_t)i0 * (k == 9 ? ts : es);
        c->link_slot_base = c->d_counts + s;
        c->link_parent_base = i0;
        int rc = picsarqed_qed_step(c, species, dtype, tau_dtype, m, ds[0], ds[1], ds[2], ds[3], ds[4], ds[5], ds[6],
                                    ds[7], ds[8], ds[9], dt, seed, step, id_base + (unsigned long long)i0, capacity,
                                    d_sec_p[0], d_sec_p[1], d_sec_p[2], d_sec_tau[0], d_sec_p[3], d_sec_p[4],
                                    d_sec_p[5], d_sec_tau[1], h_parent ? d_parent : nullptr, c->d_counts + s + 1);
        if (rc) return rc;
        PXQ_CUDA(c, cudaEventRecord(stepped, c->stream));
        PXQ_CUDA(c, cudaStreamWaitEvent(c->d2h_stream, stepped, 0));
        for (int k = 0; k < 4; ++k) {
            const size_t w = k == 3 ? ts : es;
            PXQ_CUDA(c, cudaMemcpyAsync(static_cast<char*>(h_back[k]) + (size_t)i0 * w,
                                        static_cast<const char*>(d[back_of[k]]) + (size_t)i0 * w, (size_t)m * w,
                                        cudaMemcpyDeviceToHost, c->d2h_stream));
        }
    }
    PXQ_CUDA(c, cudaMemcpyAsync(c->h_counts, c->d_counts + n_slabs, sizeof(unsigned long long), cudaMemcpyDeviceToHost,
                                c->stream));
    PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    *h_n_out = c->h_counts[0];
    const size_t m = (size_t)std::min<unsigned long long>(*h_n_out, (unsigned long long)capacity);
    if (m > 0 && h_sec) {
        // order of h_sec: leptons: ph px,py,pz,tau; photons: el px,py,pz,tau, po px,py,pz,tau
        if (species == 0) {
            for (int k = 0; k < 3; ++k)
                PXQ_CUDA(c, cudaMemcpyAsync(h_sec[k], d_sec_p[k], m * es, cudaMemcpyDeviceToHost, c->stream));
            PXQ_CUDA(c, cudaMemcpyAsync(h_sec[3], d_sec_tau[0], m * ts, cudaMemcpyDeviceToHost, c->stream));
        } else {
            for (int s = 0; s < 2; ++s) {
                for (int k = 0; k < 3; ++k)
                    PXQ_CUDA(c, cudaMemcpyAsync(h_sec[4 * s + k], d_sec_p[3 * s + k], m * es, cudaMemcpyDeviceToHost, c->stream));
                PXQ_CUDA(c, cudaMemcpyAsync(h_sec[4 * s + 3], d_sec_tau[s], m * ts, cudaMemcpyDeviceToHost, c->stream));
            }
        }
        if (h_parent) PXQ_CUDA(c, cudaMemcpyAsync(h_parent, d_parent, m * sizeof(long long), cudaMemcpyDeviceToHost, c->stream));
        PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    PXQ_CUDA(c, cudaStreamSynchronize(c->d2h_stream));
    return PICSARQED_OK;
}

extern "C" int picsarqed_build_tables(picsarqed_ctx* c, const picsarqed_table_params* p) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (!params_ok(p)) return fail(c, PICSARQED_ERR_INVALID, "bad table parameters");
    if ((size_t)std::max(p->qs_n_xi, p->bw_n_xi) * sizeof(double) > 200 * 1024)
        return fail(c, PICSARQED_ERR_INVALID, "n_xi too large for the row builder (max 25600)");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    c->have_tables = false;
    if (int rc = alloc_tables(c, *p)) return rc;
    // The two processes are independent: they are built on two streams, so that a small table set (256 rows each for 148
    // SMs) fills the GPU.  A 2D table with its own row count is a second launch of the same kernel: rows without the 1D
    // value, then the 1D values without rows.
    if (!c->aux_stream) PXQ_CUDA(c, cudaStreamCreateWithFlags(&c->aux_stream, cudaStreamNonBlocking));
    if (!c->aux_event[0])
        for (int k = 0; k < 2; ++k) PXQ_CUDA(c, cudaEventCreateWithFlags(&c->aux_event[k], cudaEventDisableTiming));
    if (!c->build_event[0])
        for (int k = 0; k < 2; ++k) PXQ_CUDA(c, cudaEventCreate(&c->build_event[k]));
    PXQ_CUDA(c, cudaEventRecord(c->build_event[0], c->stream));
    PXQ_CUDA(c, cudaEventRecord(c->aux_event[0], c->stream));            // (the tables were just cleared on c->stream)
    PXQ_CUDA(c, cudaStreamWaitEvent(c->aux_stream, c->aux_event[0], 0));
    for (int kind = 0; kind < 2; ++kind) {
        cudaStream_t st = kind == 0 ? c->stream : c->aux_stream;
        const int n1 = kind == 0 ? p->qs_n_chi : p->bw_n_chi, n2 = rows_2d(*p, kind);
        TableBuildArgs a;
        a.chi_min = kind == 0 ? p->qs_chi_min : p->bw_chi_min;
        a.chi_max = kind == 0 ? p->qs_chi_max : p->bw_chi_max;
        a.n_xi = kind == 0 ? p->qs_n_xi : p->bw_n_xi;
        a.xi_min = p->qs_xi_min;
        double* rows = c->tab64[kind == 0 ? PICSARQED_TAB_QS_LNP : PICSARQED_TAB_BW_P];
        double* ln1d = c->tab64[kind == 0 ? PICSARQED_TAB_LNG : PICSARQED_TAB_LNT];
        const size_t smem = (size_t)a.n_xi * sizeof(double);
        auto launch = [&](int n_chi, double* r, double* l) -> cudaError_t {
            a.n_chi = n_chi;
            a.rows = r;
            a.ln1d = l;
            if (kind == 0) {
                if (smem > 48 * 1024) cudaFuncSetAttribute(table_rows_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
                table_rows_kernel<0><<<n_chi, kTabThreads, smem, st>>>(a);
            } else {
                if (smem > 48 * 1024) cudaFuncSetAttribute(table_rows_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
                table_rows_kernel<1><<<n_chi, kTabThreads, smem, st>>>(a);
            }
            return cudaGetLastError();
        };
        if (n1 == n2) {
            PXQ_CUDA(c, launch(n1, rows, ln1d));
        } else {
            PXQ_CUDA(c, launch(n2, rows, nullptr));
            // the 1D values alone: the row total does not need the table's columns -- the cell routines cut every cell
            // into panels over which the integrand varies by a bounded factor, so 64 wide cells cost a thirtieth of 2048
            // narrow ones and give the same integral (to ~1e-12; the two differ only in where the panels end)
            a.n_xi = std::min(a.n_xi, 64);
            PXQ_CUDA(c, launch(n1, nullptr, ln1d));
        }
    }
    PXQ_CUDA(c, cudaEventRecord(c->aux_event[1], c->aux_stream));
    PXQ_CUDA(c, cudaStreamWaitEvent(c->stream, c->aux_event[1], 0));
    PXQ_CUDA(c, cudaEventRecord(c->build_event[1], c->stream));          // (the quadrature kernels of both processes end here)
    if (int rc = narrow_tables(c)) return rc;
    if (int rc = build_guides(c)) return rc;
    PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    float ms = 0.f;
    PXQ_CUDA(c, cudaEventElapsedTime(&ms, c->build_event[0], c->build_event[1]));
    c->build_ms = ms;
    c->have_tables = true;
    return PICSARQED_OK;
}

extern "C" int picsarqed_get_table_build_ms(picsarqed_ctx* c, double* host_ms) {
    if (!c || !host_ms) return PICSARQED_ERR_INVALID;
    *host_ms = c->build_ms;
    return PICSARQED_OK;
}

// =====================================================================================
//  closed loop in a uniform field (cascade.cuh)
// =====================================================================================
extern "C" int picsarqed_boris_push_uniform(picsarqed_ctx* c, int dtype, long long n, void* px, void* py, void* pz,
                                            int charge_sign, const double* e, const double* b, double dt) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (c->unit_system != PICSARQED_UNITS_LIBRARY)
        return fail(c, PICSARQED_ERR_INVALID, "the closed-loop calls take the library's own units");
    if (n < 0 || (charge_sign != 1 && charge_sign != -1) || !e || !b)
        return fail(c, PICSARQED_ERR_INVALID, "bad n, charge_sign, e or b");
    if (dtype != PICSARQED_F64 && dtype != PICSARQED_F32) return fail(c, PICSARQED_ERR_DTYPE, "bad dtype");
    if (n == 0) return PICSARQED_OK;
    const void* a[3] = {px, py, pz};
    if (int rc = check_arrays(c, a, 3)) return rc;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    BorisArgs args;
    const double k = charge_sign * dt * kInvTauC * 0.5;
    for (int j = 0; j < 3; ++j) {
        args.ke[j] = k * e[j];
        args.kb[j] = k * b[j];
    }
    if (dtype == PICSARQED_F64)
        boris_kernel<double><<<stream_grid(c, (n + 1) / 2, 256), 256, 0, c->stream>>>((double*)px, (double*)py, (double*)pz, n, args);
    else
        boris_kernel<float><<<stream_grid(c, (n + 3) / 4, 256), 256, 0, c->stream>>>((float*)px, (float*)py, (float*)pz, n, args);
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

extern "C" int picsarqed_set_chi_threshold(picsarqed_ctx* c, double chi_min) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (!(chi_min >= 0.0) || !std::isfinite(chi_min)) return fail(c, PICSARQED_ERR_INVALID, "set_chi_threshold: chi_min must be >= 0");
    c->chi_event_min = chi_min;
    return PICSARQED_OK;
}

extern "C" int picsarqed_classical_loss(picsarqed_ctx* c, int dtype, long long n, void* px, void* py, void* pz, const void* ex,
                                        const void* ey, const void* ez, const void* bx, const void* by, const void* bz,
                                        double dt) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (c->unit_system != PICSARQED_UNITS_LIBRARY)
        return fail(c, PICSARQED_ERR_INVALID, "the closed-loop calls take the library's own units");
    if (n < 0) return fail(c, PICSARQED_ERR_INVALID, "bad n");
    if (dtype != PICSARQED_F64 && dtype != PICSARQED_F32) return fail(c, PICSARQED_ERR_DTYPE, "bad dtype");
    if (n == 0 || c->chi_event_min == 0.0) return PICSARQED_OK;
    const void* a[9] = {px, py, pz, ex, ey, ez, bx, by, bz};
    if (int rc = check_arrays(c, a, 9)) return rc;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    const double c2_min = c->chi_event_min * c->chi_event_min, loss_dt = (2.0 / 3.0) * kAlphaOverTauC * dt;
    if (dtype == PICSARQED_F64)
        classical_loss_kernel<double><<<stream_grid(c, (n + 1) / 2, 256), 256, 0, c->stream>>>(
            (double*)px, (double*)py, (double*)pz, (const double*)ex, (const double*)ey, (const double*)ez, (const double*)bx,
            (const double*)by, (const double*)bz, n, c2_min, loss_dt);
    else
        classical_loss_kernel<float><<<stream_grid(c, (n + 3) / 4, 256), 256, 0, c->stream>>>(
            (float*)px, (float*)py, (float*)pz, (const float*)ex, (const float*)ey, (const float*)ez, (const float*)bx,
            (const float*)by, (const float*)bz, n, c2_min, loss_dt);
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

extern "C" int picsarqed_append_secondaries(picsarqed_ctx* c, int dtype, int tau_dtype, long long m_max, const void* s_px,
                                            const void* s_py, const void* s_pz, const void* s_tau,
                                            const unsigned long long* d_count, double min_energy, void* d_px, void* d_py,
                                            void* d_pz, void* d_tau, long long dst_n, long long dst_capacity,
                                            unsigned long long* d_new_n) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (m_max < 0 || dst_n < 0 || dst_capacity < dst_n || !d_count || !d_new_n || !(min_energy >= 0.0))
        return fail(c, PICSARQED_ERR_INVALID, "bad m_max, dst_n, dst_capacity, min_energy, d_count or d_new_n");
    PXQ_CUDA(c, cudaSetDevice(c->device));
    if (m_max == 0) {
        const unsigned long long v = (unsigned long long)dst_n;
        PXQ_CUDA(c, cudaMemcpyAsync(d_new_n, &v, sizeof(v), cudaMemcpyHostToDevice, c->stream));
        PXQ_CUDA(c, cudaStreamSynchronize(c->stream));  // (v lives on this stack frame)
        return PICSARQED_OK;
    }
    const void* chk[8] = {s_px, s_py, s_pz, s_tau, d_px, d_py, d_pz, d_tau};
    if (int rc = check_arrays(c, chk, 8)) return rc;
    const void* s_p[3] = {s_px, s_py, s_pz};
    void* d_p[3] = {d_px, d_py, d_pz};
    PXQ_DISPATCH_RT(c, dtype, tau_dtype,
                    return (launch_append<R, TR>(c, m_max, s_p, s_tau, d_count, min_energy, d_p, d_tau, dst_n, nullptr,
                                                 dst_capacity, c->d_cas + 15, d_new_n)));
}

extern "C" int picsarqed_energy_spectrum(picsarqed_ctx* c, int species, int dtype, long long n, const void* px,
                                         const void* py, const void* pz, double e_min, double e_max, int nbins,
                                         unsigned long long* hist) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (c->unit_system != PICSARQED_UNITS_LIBRARY)
        return fail(c, PICSARQED_ERR_INVALID, "the closed-loop calls take the library's own units");
    if (n < 0 || (species != 0 && species != 1) || !(e_min > 0.0) || !(e_max > e_min) || nbins < 1 ||
        nbins > kSpectrumMaxBins || !hist)
        return fail(c, PICSARQED_ERR_INVALID, "bad n, species, energy range, nbins or hist");
    if (dtype != PICSARQED_F64 && dtype != PICSARQED_F32) return fail(c, PICSARQED_ERR_DTYPE, "bad dtype");
    if (n == 0) return PICSARQED_OK;
    const void* a[3] = {px, py, pz};
    if (int rc = check_arrays(c, a, 3)) return rc;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    const double ln_min = std::log(e_min), scale = nbins / (std::log(e_max) - std::log(e_min));
    const int grid = (int)std::max<long long>(1, std::min<long long>((n + 1023) / 1024, (long long)c->num_sms * 8));
    const size_t smem = (size_t)nbins * sizeof(unsigned int);
#define PXQ_SPECTRUM(R, S)                                                                                     \
    spectrum_kernel<R, S><<<grid, 256, smem, c->stream>>>((const R*)px, (const R*)py, (const R*)pz, n, ln_min, \
                                                          scale, nbins, hist)
    if (dtype == PICSARQED_F64) {
        if (species == 0) PXQ_SPECTRUM(double, 0); else PXQ_SPECTRUM(double, 1);
    } else {
        if (species == 0) PXQ_SPECTRUM(float, 0); else PXQ_SPECTRUM(float, 1);
    }
#undef PXQ_SPECTRUM
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

extern "C" int picsarqed_cascade_step(picsarqed_ctx* c, int dtype, int tau_dtype, picsarqed_species_arrays* el,
                                      picsarqed_species_arrays* po, picsarqed_species_arrays* ph, const double* e,
                                      const double* b, double dt, unsigned long long seed, unsigned long long step,
                                      double photon_min_energy, int push, unsigned long long* h_events) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (c->unit_system != PICSARQED_UNITS_LIBRARY)
        return fail(c, PICSARQED_ERR_INVALID, "the closed-loop calls take the library's own units");
    if (!el || !po || !ph || !e || !b || !(photon_min_energy >= 0.0))
        return fail(c, PICSARQED_ERR_INVALID, "null species, e or b, or bad photon_min_energy");
    if ((dtype != 0 && dtype != 1) || (tau_dtype != 0 && tau_dtype != 1) || (dtype == 1 && tau_dtype == 0))
        return fail(c, PICSARQED_ERR_DTYPE, "unsupported (dtype, tau_dtype) combination");
    picsarqed_species_arrays* sp[3] = {el, po, ph};
    for (int k = 0; k < 3; ++k)
        if (sp[k]->n < 0 || sp[k]->capacity < sp[k]->n) return fail(c, PICSARQED_ERR_INVALID, "species: bad n or capacity");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    {
        // the Philox counter holds the species only as lepton / photon: an electron and a positron with the
        // same id would draw the same numbers, so the two arrays must own disjoint id ranges (R21: 0 and 2^40)
        const unsigned long long e0 = el->id_base, e1 = e0 + (unsigned long long)el->capacity;
        const unsigned long long p0 = po->id_base, p1 = p0 + (unsigned long long)po->capacity;
        if (el->capacity > 0 && po->capacity > 0 && e0 < p1 && p0 < e1)
            return fail(c, PICSARQED_ERR_INVALID, "cascade_step: the id ranges [id_base, id_base + capacity) of electrons and positrons overlap");
    }
    PXQ_CUDA(c, cudaSetDevice(c->device));
    const size_t es = dtype ? 8 : 4, ts = tau_dtype ? 8 : 4;
    auto pad = [](size_t x) { return (x + 255) & ~(size_t)255; };
    const long long n_e = el->n, n_p = po->n, n_g = ph->n;
    const long long n_max = std::max(n_e, std::max(n_p, n_g));
    // scratch: six constant field arrays of n_field entries; secondary buffers (photons of the electrons, photons of
    // the positrons, electrons and positrons of the photons), 3 momenta + tau each
    auto need_for = [&](long long nf, long long ne, long long np, long long ng) {
        return 6 * pad((size_t)nf * es) + (3 * pad((size_t)ne * es) + pad((size_t)ne * ts)) +
               (3 * pad((size_t)np * es) + pad((size_t)np * ts)) + 2 * (3 * pad((size_t)ng * es) + pad((size_t)ng * ts));
    };
    long long n_field = std::max<long long>(c->cas_field_n, n_max);
    if (need_for(n_field, n_e, n_p, n_g) > c->cas_bytes) {  // grow with headroom: populations rise step after step
        n_field = n_max + n_max / 2 + 1024;
        const size_t want = need_for(n_field, n_e + n_e / 2 + 1024, n_p + n_p / 2 + 1024, n_g + n_g / 2 + 1024);
        PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
        if (c->cas) cudaFree(c->cas);
        c->cas = nullptr;
        c->cas_bytes = 0;
        c->cas_field_n = 0;
        PXQ_CUDA(c, cudaMalloc(&c->cas, want));
        c->cas_bytes = want;
    }
    char* base = static_cast<char*>(c->cas);
    void* f[6];
    for (int k = 0; k < 6; ++k) f[k] = base + k * pad((size_t)n_field * es);
    char* q = base + 6 * pad((size_t)n_field * es);
    auto carve = [&](long long m, void** p4) {  // 3 momenta + tau of m entries
        for (int k = 0; k < 3; ++k) { p4[k] = q; q += pad((size_t)m * es); }
        p4[3] = q;
        q += pad((size_t)m * ts);
    };
    void *ph_e[4], *ph_p[4], *pair_e[4], *pair_p[4];
    carve(n_e, ph_e);
    carve(n_p, ph_p);
    carve(n_g, pair_e);
    carve(n_g, pair_p);
    const double fv[6] = {e[0], e[1], e[2], b[0], b[1], b[2]};
    bool same = c->cas_field_dtype == dtype && c->cas_field_n >= n_field;
    for (int k = 0; k < 6; ++k) same = same && c->cas_field[k] == fv[k];
    if (!same && n_field > 0) {
        for (int k = 0; k < 6; ++k) {
            const int grid = stream_grid(c, n_field, 256);
            if (dtype) fill_kernel<double><<<grid, 256, 0, c->stream>>>((double*)f[k], n_field, fv[k]);
            else fill_kernel<float><<<grid, 256, 0, c->stream>>>((float*)f[k], n_field, (float)fv[k]);
            c->cas_field[k] = fv[k];
        }
        PXQ_CUDA(c, cudaGetLastError());
        c->cas_field_n = n_field;
        c->cas_field_dtype = dtype;
    }
    // d_cas: [0..2] events of electrons, positrons, photons; [3] photons before the appends, [4] after the first,
    // [5] after the second; [6] electrons, [7] positrons after the pairs; [15] scratch (kept count of an append)
    PXQ_CUDA(c, cudaMemsetAsync(c->d_cas, 0, 16 * sizeof(unsigned long long), c->stream));
    if (push) {
        if (int rc = picsarqed_boris_push_uniform(c, dtype, n_e, el->px, el->py, el->pz, -1, e, b, dt)) return rc;
        if (int rc = picsarqed_boris_push_uniform(c, dtype, n_p, po->px, po->py, po->pz, +1, e, b, dt)) return rc;
    }
    if (c->chi_event_min > 0.0) {   // below the threshold the leptons radiate classically (R24)
        if (int rc = picsarqed_classical_loss(c, dtype, n_e, el->px, el->py, el->pz, f[0], f[1], f[2], f[3], f[4], f[5], dt)) return rc;
        if (int rc = picsarqed_classical_loss(c, dtype, n_p, po->px, po->py, po->pz, f[0], f[1], f[2], f[3], f[4], f[5], dt)) return rc;
    }
    if (n_e > 0)
        if (int rc = picsarqed_qed_step(c, 0, dtype, tau_dtype, n_e, el->px, el->py, el->pz, f[0], f[1], f[2], f[3], f[4], f[5],
                                        el->tau, dt, seed, step, el->id_base, n_e, ph_e[0], ph_e[1], ph_e[2], ph_e[3],
                                        nullptr, nullptr, nullptr, nullptr, nullptr, c->d_cas + 0))
            return rc;
    if (n_p > 0)
        if (int rc = picsarqed_qed_step(c, 0, dtype, tau_dtype, n_p, po->px, po->py, po->pz, f[0], f[1], f[2], f[3], f[4], f[5],
                                        po->tau, dt, seed, step, po->id_base, n_p, ph_p[0], ph_p[1], ph_p[2], ph_p[3],
                                        nullptr, nullptr, nullptr, nullptr, nullptr, c->d_cas + 1))
            return rc;
    if (n_g > 0)
        if (int rc = picsarqed_qed_step(c, 1, dtype, tau_dtype, n_g, ph->px, ph->py, ph->pz, f[0], f[1], f[2], f[3], f[4], f[5],
                                        ph->tau, dt, seed, step, ph->id_base, n_g, pair_e[0], pair_e[1], pair_e[2],
                                        pair_e[3], pair_p[0], pair_p[1], pair_p[2], pair_p[3], nullptr, c->d_cas + 2))
            return rc;
    // feed back (R20): photons of the electrons, then of the positrons; then the pairs
    c->h_cas[0] = (unsigned long long)n_g;  // (pinned; not read back before the synchronize below)
    for (int k = 3; k <= 5; ++k)
        PXQ_CUDA(c, cudaMemcpyAsync(c->d_cas + k, c->h_cas, 8, cudaMemcpyHostToDevice, c->stream));
    void* ph_dst[3] = {ph->px, ph->py, ph->pz};
    void* el_dst[3] = {el->px, el->py, el->pz};
    void* po_dst[3] = {po->px, po->py, po->pz};
    // (an append never reads and writes the same counter: every block reads its start while block 0 writes the end)
#define PXQ_APPEND(SRC, M, CNT, THR, DST, DTAU, DSTN, DSTN_PTR, CAP, OUT)                                              \
    do {                                                                                                               \
        if ((M) > 0) {                                                                                                 \
            PXQ_DISPATCH_RT(c, dtype, tau_dtype, {                                                                     \
                if (int rc = launch_append<R, TR>(c, (M), SRC, SRC[3], (CNT), (THR), DST, DTAU, (DSTN), (DSTN_PTR),    \
                                                  (CAP), c->d_cas + 15, (OUT)))                                        \
                    return rc;                                                                                         \
            });                                                                                                        \
        }                                                                                                              \
    } while (0)
    PXQ_APPEND(ph_e, n_e, c->d_cas + 0, photon_min_energy, ph_dst, ph->tau, 0, c->d_cas + 3, ph->capacity, c->d_cas + 4);
    PXQ_APPEND(ph_p, n_p, c->d_cas + 1, photon_min_energy, ph_dst, ph->tau, 0, c->d_cas + 4, ph->capacity, c->d_cas + 5);
    PXQ_APPEND(pair_e, n_g, c->d_cas + 2, 0.0, el_dst, el->tau, n_e, nullptr, el->capacity, c->d_cas + 6);
    PXQ_APPEND(pair_p, n_g, c->d_cas + 2, 0.0, po_dst, po->tau, n_p, nullptr, po->capacity, c->d_cas + 7);
#undef PXQ_APPEND
    PXQ_CUDA(c, cudaMemcpyAsync(c->h_cas, c->d_cas, 8 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    PXQ_CUDA(c, cudaStreamSynchronize(c->stream));
    if (h_events)
        for (int k = 0; k < 3; ++k) h_events[k] = c->h_cas[k];
    const long long new_n[3] = {n_g > 0 ? (long long)c->h_cas[6] : n_e, n_g > 0 ? (long long)c->h_cas[7] : n_p,
                                (long long)(n_p > 0 ? c->h_cas[5] : c->h_cas[4])};
    bool overflow = false;
    for (int k = 0; k < 3; ++k) {
        overflow = overflow || new_n[k] > sp[k]->capacity;
        sp[k]->n = std::min(new_n[k], sp[k]->capacity);
    }
    if (overflow) return fail(c, PICSARQED_ERR_INVALID, "cascade_step: a species exceeded its capacity");
    return PICSARQED_OK;
}

// =====================================================================================
//  table functions per value (lookup.cuh)
// =====================================================================================
extern "C" int picsarqed_table_function(picsarqed_ctx* c, int kind, int dtype, long long n, const void* chi, void* out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || (kind != 0 && kind != 1)) return fail(c, PICSARQED_ERR_INVALID, "bad n or kind");
    if (dtype != PICSARQED_F64 && dtype != PICSARQED_F32) return fail(c, PICSARQED_ERR_DTYPE, "bad dtype");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    if (n == 0) return PICSARQED_OK;
    const void* a[2] = {chi, out};
    if (int rc = check_arrays(c, a, 2)) return rc;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    const int grid = stream_grid(c, n, 256);
#define PXQ_TF(R, K) table_function_kernel<R, K><<<grid, 256, 0, c->stream>>>((const R*)chi, (R*)out, n, view_1d<R>(c, K))
    if (dtype == PICSARQED_F64) {
        if (kind == 0) PXQ_TF(double, 0); else PXQ_TF(double, 1);
    } else {
        if (kind == 0) PXQ_TF(float, 0); else PXQ_TF(float, 1);
    }
#undef PXQ_TF
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}

extern "C" int picsarqed_sample_xi(picsarqed_ctx* c, int kind, int dtype, long long n, const void* chi, const void* r,
                                   void* xi_out) {
    if (!c) return PICSARQED_ERR_INVALID;
    if (n < 0 || (kind != 0 && kind != 1)) return fail(c, PICSARQED_ERR_INVALID, "bad n or kind");
    if (dtype != PICSARQED_F64 && dtype != PICSARQED_F32) return fail(c, PICSARQED_ERR_DTYPE, "bad dtype");
    if (!c->have_tables) return fail(c, PICSARQED_ERR_NO_TABLES, "no tables: call build_tables or import_tables");
    if (n == 0) return PICSARQED_OK;
    const void* a[3] = {chi, r, xi_out};
    if (int rc = check_arrays(c, a, 3)) return rc;
    PXQ_CUDA(c, cudaSetDevice(c->device));
    const int grid = stream_grid(c, n, 256);
#define PXQ_SX(R, K) \
    sample_xi_kernel<R, K><<<grid, 256, 0, c->stream>>>((const R*)chi, (const R*)r, (R*)xi_out, n, view_2d<R>(c, K))
    if (dtype == PICSARQED_F64) {
        if (kind == 0) PXQ_SX(double, 0); else PXQ_SX(double, 1);
    } else {
        if (kind == 0) PXQ_SX(float, 0); else PXQ_SX(float, 1);
    }
#undef PXQ_SX
    PXQ_CUDA(c, cudaGetLastError());
    return PICSARQED_OK;
}
