/* =====================================================================================
 *  picsarqed.h -- C ABI of the B200-native PICSAR-QED hot path (arXiv 2110.00256).
 *
 *  The library (paper_2110_00256_b200/libpicsarqed.so) is hand-written CUDA for sm_100a.
 *  Citations are PAPER.md:<line> of the paper text.  DESIGN.md lists how garbled or silent
 *  passages were read (R1..R16) and the data layout.
 *
 *  Conventions
 *  -----------
 *  * Every entry point returns an int status: PICSARQED_OK or one of the error codes below.
 *    No C++ exception crosses the boundary.  picsarqed_last_error() returns a text for the
 *    last non-OK status of that context.
 *  * DEVICE pointers: all particle, field, optical-depth, secondary and counter arguments
 *    (anything called px..bz, tau, *_out, ph_*, el_*, po_*, parent, d_*).  They are owned by
 *    the caller (e.g. torch allocations), structure-of-arrays, contiguous, 16-byte aligned;
 *    the library never allocates, frees or keeps them.  Work is enqueued on the context's
 *    stream and the call returns without synchronising, except where stated.
 *  * HOST pointers: picsarqed_table_params, the table arrays of import/export, every
 *    argument whose name starts with host_ or h_, and every argument of the *_host calls.
 *  * Units: momentum p in m_e c; fields e = E/E_s, b = cB/E_s with E_s the Schwinger field
 *    (eq.1); dt in seconds.  The tables are adimensional.
 *  * dtype / tau_dtype: PICSARQED_F32 or PICSARQED_F64 -- element type of the particle/field
 *    arrays and of the optical-depth arrays (configuration 5 of BASELINE.json mixes fp32
 *    particles with fp64 optical depth).  fp32 particle arithmetic reads the fp32-rounded
 *    copy of the tables ("computed in double, stored in single").
 *  * species: PICSARQED_LEPTON (electron or positron: eq.2 and eq.15 do not depend on the
 *    sign of the charge) or PICSARQED_PHOTON.
 *  * Random numbers: Philox4x32-10, key = seed, counter = (particle id, step, purpose,
 *    species); particle id = id_base + array index.  See DESIGN.md "RNG".
 * ===================================================================================== */
#ifndef PICSARQED_H
#define PICSARQED_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PICSARQED_OK 0
#define PICSARQED_ERR_INVALID 1  /* null/misaligned pointer, n < 0, bad enum, bad table params */
#define PICSARQED_ERR_CUDA 2     /* a CUDA runtime call failed; see picsarqed_last_error        */
#define PICSARQED_ERR_NO_TABLES 4 /* build_tables / import_tables has not been called           */
#define PICSARQED_ERR_DTYPE 5    /* unsupported dtype combination                              */
/* There is no "capacity exceeded" status (SURVEY.md 8(b) proposed an all-or-nothing status 3): when more particles fire than
 * the output buffers hold, the first `capacity` fired parents (in index order) are processed, the later ones are left
 * exactly as the evolve pass left them (optical depth still negative, momentum untouched) and *d_n_out receives the TOTAL
 * number that fired, so the caller sees the overflow by comparing it with `capacity` and can run generate_* again on the
 * same arrays with fresh buffers (R16). */

#define PICSARQED_F32 0
#define PICSARQED_F64 1
#define PICSARQED_LEPTON 0
#define PICSARQED_PHOTON 1

/* which table, for export: */
#define PICSARQED_TAB_LNG 0    /* ln G(chi_i),           n = qs_n_chi     */
#define PICSARQED_TAB_QS_LNP 1 /* ln P_QS[chi_n][xi_m],  n = rows*qs_n_xi, row-major; rows = qs_n_chi_2d or qs_n_chi */
#define PICSARQED_TAB_LNT 2    /* ln T(chi_gamma,i),     n = bw_n_chi     */
#define PICSARQED_TAB_BW_P 3   /* P_BW[chi_n][xi_m],     n = bw_n_chi*bw_n_xi, row-major */

typedef struct picsarqed_ctx picsarqed_ctx;

/* Table geometry (the paper's benchmark set is at :301).
 * chi grids are log-spaced and include both ends; QS xi_m = xi_min^(1 - m/(n_xi-1)) on
 * [xi_min, 1]; BW xi_m = 0.5 m/(n_xi-1) on [0, 1/2] (the other half follows from
 * P(xi) = 1 - P(1-xi)).  All counts >= 2; 0 < min < max; 0 < qs_xi_min < 1. */
typedef struct {
    double qs_chi_min, qs_chi_max;
    int qs_n_chi;
    double qs_xi_min;
    int qs_n_xi;
    double bw_chi_min, bw_chi_max;
    int bw_n_chi;
    int bw_n_xi;
    /* Rows of the two 2D tables when they differ from the 1D counts above (BASELINE configuration 4: 4096-point 1D
     * tables with 2048 x 2048 CDF tables): log-spaced on the same [chi_min, chi_max], both ends included.  0 = the same
     * grid as the 1D table (the paper's own sets). */
    int qs_n_chi_2d;
    int bw_n_chi_2d;
} picsarqed_table_params;

/* ---- context ------------------------------------------------------------------------
 * One context per (device, stream).  cuda_stream is a cudaStream_t passed as void* (0 = the
 * legacy default stream).  The context owns the tables and a few KB of scan scratch. */
int picsarqed_create(picsarqed_ctx** out, int cuda_device, void* cuda_stream);
int picsarqed_destroy(picsarqed_ctx* ctx);
const char* picsarqed_last_error(const picsarqed_ctx* ctx);
/* bit 0: library was compiled for sm_100a; returns the CUDA runtime version in the upper bits */
int picsarqed_version(void);
/* Tuning knobs (integers): "evolve_unroll" in {0 (default), 1, 2, 4} = independent 128-bit
 * loads per array per thread in the evolve kernel; "evolve_ctas_per_sm" (0 = occupancy limit);
 * "event_config" 0..1 = shape of the event kernel; "time_kernels" 0/1; "stage_records" 0/1 (see
 * evolve_optical_depth); "fused_step" 0/1 = qed_step as one warp-specialised kernel (experimental, slower today: DESIGN.md 11),
 * with "step_config", "step_spill", "step_batch_wait" its tuning knobs;
 * "event_pdl" 0/1 (default 1) = the event kernel is launched as a programmatic dependent of the offsets scan (its CTAs become
 * resident while the scan runs and wait for it at griddepcontrol.wait);
 * "evolve_redraw" 0..2 = which pass of qed_step re-draws the optical depth of the leptons that emit (same Philox words, same
 * value either way): 0 = the event pass (a fourth scattered store per event), 1 = the evolve pass for fp64 particles, 2 (default)
 * = the evolve pass for every dtype (the new value leaves with the pass's own vector store);
 * "host_slabs" 0..64 = number of slabs step_host pipelines (0 = automatic: slabs of at least
 * 2^20 particles, at most 32; 1 = copy in, step, copy out, one after the other). */
int picsarqed_set_option(picsarqed_ctx* ctx, const char* name, long long value);
/* ---- unit systems --------------------------------------------------------
 * The library's own units: momenta in m_e c, E in E_s = m_e^2 c^3/(q_e hbar), B in E_s/c, times in
 * seconds.  set_units declares the unit system of the CALLER's arrays for chi,
 * evolve_optical_depth, generate_photons, generate_pairs, qed_step, step_host and schwinger_rate:
 * momenta and fields are scaled in registers where they are loaded, momenta back where they are
 * stored (no extra pass over memory); dt is taken in the system's time unit.  Tables are
 * adimensional and serve every system.  The closed-loop calls take the library's units only.
 *   LIBRARY      the default
 *   SI           kg m/s, V/m, T, s
 *   NORM_OMEGA   c = q_e = m_e = 1 with a reference angular frequency `reference` [1/s]: p in m_e c,
 *                E in m_e c omega/q_e, B in m_e omega/q_e, t in 1/omega
 *   NORM_LAMBDA  the same with a reference length `reference` [m] (omega = c/lambda)
 *   HL_MEV       Heaviside-Lorentz natural units (hbar = c = 1) with 1 MeV: p in MeV, E and B in MeV^2,
 *                t in 1/MeV (the paper's internal system)
 * get_unit_scales writes the four multipliers (p, E, B, t) that take the caller's values to the
 * library's units. */
#define PICSARQED_UNITS_LIBRARY 0
#define PICSARQED_UNITS_SI 1
#define PICSARQED_UNITS_NORM_OMEGA 2
#define PICSARQED_UNITS_NORM_LAMBDA 3
#define PICSARQED_UNITS_HL_MEV 4
int picsarqed_set_units(picsarqed_ctx* ctx, int system, double reference);
int picsarqed_get_unit_scales(picsarqed_ctx* ctx, double* scales /* host, 4 doubles */);

/* With "time_kernels" = 1 every qed_step brackets its evolve pass and its event pass (offsets scan +
 * event kernel) with CUDA events on the context's stream.  get_timing synchronises, writes the
 * accumulated milliseconds host_ms[0] (evolve pass) and host_ms[1] (event pass) and the number of
 * qed_step calls they cover, and resets the accumulation. */
int picsarqed_get_timing(picsarqed_ctx* ctx, double* host_ms, long long* host_calls);

/* ---- tables -------------------------------------------------------------------------
 * build_tables: integrates on the GPU, in fp64,
 *     T(chi_gamma) = 1/(pi sqrt3 chi_gamma) int_0^1 f_BW dxi          (eq.9)
 *     P_BW(chi_gamma, xi) = int_0^xi f_BW / int_0^1 f_BW               (eq.11)
 *     G(chi) = int_0^1 S(chi,xi)/xi dxi                                (eq.16)
 *     P_QS(chi, xi) = int_0^xi S/u du / G                              (eq.18)
 * from the K_{1/3}, K_{2/3} Bessel quadratures, and stores ln T, ln G, P_BW and ln P_QS
 * in fp64 plus an fp32-rounded copy.  Synchronises.
 * Accuracy: fixed by the scheme (panelled 8-point Gauss-Legendre over trapezoid-rule Bessel integrals), about 1e-11
 * relative on T, G, P against the oracle's adaptive quadrature; there is no tolerance knob.  n_xi <= 25600. */
int picsarqed_build_tables(picsarqed_ctx* ctx, const picsarqed_table_params* host_params);
/* Device time of the quadrature kernels of the last build_tables (CUDA events on the context's stream around the two
 * processes' launches; milliseconds).  The call's wall time adds allocation, the fp32 copies and the search guides. */
int picsarqed_get_table_build_ms(picsarqed_ctx* ctx, double* host_ms);
/* Copies table `which` to host memory as fp64 (n_elems must equal the table's size).  Synchronises. */
int picsarqed_export_tables(picsarqed_ctx* ctx, int which, double* host_dst, size_t n_elems);
/* Replaces the tables by caller-provided values (host, fp64, layouts as above).  Synchronises. */
int picsarqed_import_tables(picsarqed_ctx* ctx, const picsarqed_table_params* host_params,
                            const double* host_lnG, const double* host_qs_lnP,
                            const double* host_lnT, const double* host_bw_P);

/* ---- chi (PAPER.md:70 eq.2 leptons, :77 eq.3 photons) --------------------------------
 * chi_out[i] = sqrt(|g e + p x b|^2 - (p.e)^2), g = sqrt(1+p^2) (lepton) or |p| (photon).
 * n = 0 is a no-op. */
int picsarqed_chi(picsarqed_ctx* ctx, int species, int dtype, long long n,
                  const void* px, const void* py, const void* pz,
                  const void* ex, const void* ey, const void* ez,
                  const void* bx, const void* by, const void* bz, void* chi_out);

/* ---- Schwinger pair production (eqs.19-22) -----------------
 * rate_out[i] (device, fp64 whatever `dtype`) = d^2N/dt dV in pairs per m^3 per s for the fields of cell i:
 * q_e^2 E_s^2/(4 pi^2 hbar^2 c) eps eta coth(pi eta/eps) exp(-pi/eps), eps, eta from the invariants
 * F = (e^2 - b^2)/2 and G = e.b (fields in units of E_s).  Pairs are created at rest. */
int picsarqed_schwinger_rate(picsarqed_ctx* ctx, int dtype, long long n,
                             const void* ex, const void* ey, const void* ez,
                             const void* bx, const void* by, const void* bz, double* rate_out);

/* ---- optical depth ----------------------------------------------
 * tau[i] = -ln U(seed, id_base+i, step 0, purpose 0, species): a draw from p(x) = exp(-x). */
int picsarqed_init_optical_depth(picsarqed_ctx* ctx, int species, int tau_dtype, long long n,
                                 unsigned long long seed, unsigned long long id_base, void* tau);

/* tau[i] <- tau[i] - dN/dt(chi_i) dt, in place, with
 *   leptons: dN/dt = (2/3)(alpha/tau_C) G(chi)/gamma          (eq.15), G by eq.27
 *            (log-log interpolation of ln G, first/last value outside the table);
 *   photons: dN/dt = (alpha/tau_C) chi_gamma T(chi_gamma)/gamma_gamma (eq.8), T by
 *            eq.23 inside the table, the Erber form of eq.10 outside (R2);
 *            photons with gamma_gamma <= 2 or tau = +inf never decay (R12).
 * *d_n_events (device, 8 bytes, may be NULL) is overwritten with the number of tau[i] < 0
 * after the update (R1).
 * Option "stage_records" = 1: the call also stages, in context scratch, the record (momentum, chi^2, index) of every
 * particle that fired, and the next generate_photons / generate_pairs call on the SAME tau pointer, n, species and
 * dtypes takes them instead of re-scanning tau and gathering the parents (the two calls then cost what qed_step costs).
 * The caller promises that momenta, fields and optical depths are not modified between the two calls; any other call
 * in between drops the staged records. */
int picsarqed_evolve_optical_depth(picsarqed_ctx* ctx, int species, int dtype, int tau_dtype, long long n,
                                   const void* px, const void* py, const void* pz,
                                   const void* ex, const void* ey, const void* ez,
                                   const void* bx, const void* by, const void* bz,
                                   double dt, void* tau, unsigned long long* d_n_events);

/* ---- events ---------------------------------------------------------------------------
 * generate_photons (eqs.28-30): every lepton with tau < 0 emits one
 * photon of energy gamma_gamma = (gamma-1) xi along its momentum, xi by inverse-CDF lookup in
 * ln P_QS; the emitter keeps its direction, loses gamma_gamma of energy and gets a fresh
 * tau = -ln U.  Photons are written densely in ASCENDING PARENT INDEX: slot s holds the
 * s-th fired lepton's photon (momentum ph_p*, optical depth ph_tau, parent index ph_parent,
 * which may be NULL).
 * Capacity rule: only the first `capacity` fired parents are processed; later ones are left
 * untouched (tau stays negative, so a second call with a fresh buffer picks them up).
 * *d_n_out (device, 8 bytes, required) is overwritten with the TOTAL number of fired
 * parents, which may exceed capacity. */
int picsarqed_generate_photons(picsarqed_ctx* ctx, int dtype, int tau_dtype, long long n,
                               void* px, void* py, void* pz, /* in/out */
                               const void* ex, const void* ey, const void* ez,
                               const void* bx, const void* by, const void* bz,
                               void* tau, /* in/out */
                               unsigned long long seed, unsigned long long step,
                               unsigned long long id_base, long long capacity,
                               void* ph_px, void* ph_py, void* ph_pz, void* ph_tau,
                               long long* ph_parent, unsigned long long* d_n_out);

/* generate_photons_noalloc: picsarqed_generate_photons for callers that must not allocate (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same operation (PAPER.md:165,
 * :255-267 eqs.28-30), same arguments, same results bit for bit, same ordering, capacity rule and d_n_out;
 * the caller still passes every input and output.  What differs is the scratch of the compaction (chunk
 * counts, tile sums, tile offsets): it is a file-scope device array of 459 264 bytes inside the library, which
 * every GPU that loads the library holds until the process exits, instead of a buffer the context grows with
 * cudaMalloc.  The call issues no cudaMalloc, cudaFree or allocating library routine: one cudaMemsetAsync of
 * the tile sums (they must start at zero; the array keeps the last call's contents) and three kernels on the
 * context's stream.  (The tables must be there already: build_tables / import_tables allocate.)
 * Limit: n <= PICSARQED_NOALLOC_MAX_N (16 Mi particles per call); a larger n returns
 * PICSARQED_ERR_INVALID with a message naming the limit, and nothing is enqueued.
 * EVERY call on a device -- from any context, any stream -- shares the one array: calls that overlap on the
 * GPU race.  Calls on one stream, or ordered by events, are safe.  If the context holds records staged by
 * evolve_optical_depth ("stage_records"), they are dropped. */
#define PICSARQED_NOALLOC_MAX_N (1ll << 24)
int picsarqed_generate_photons_noalloc(picsarqed_ctx* ctx, int dtype, int tau_dtype, long long n,
                                       void* px, void* py, void* pz, /* in/out */
                                       const void* ex, const void* ey, const void* ez,
                                       const void* bx, const void* by, const void* bz,
                                       void* tau, /* in/out */
                                       unsigned long long seed, unsigned long long step,
                                       unsigned long long id_base, long long capacity,
                                       void* ph_px, void* ph_py, void* ph_pz, void* ph_tau,
                                       long long* ph_parent, unsigned long long* d_n_out);

/* generate_pairs (eqs.24-26): every photon with tau < 0 becomes an
 * electron-positron pair, chi_-/chi_gamma = xi by inverse-CDF lookup in P_BW on
 * r' = min(r, 1-r) (r <= 1/2: the electron takes xi, else 1-xi),
 * gamma_pm = 1 + (gamma_gamma-2) xi_pm, both along the photon.  The photon is marked dead:
 * p = 0, tau = +inf.  Ordering, capacity rule and d_n_out as above. */
int picsarqed_generate_pairs(picsarqed_ctx* ctx, int dtype, int tau_dtype, long long n,
                             void* px, void* py, void* pz, /* in/out */
                             const void* ex, const void* ey, const void* ez,
                             const void* bx, const void* by, const void* bz,
                             void* tau, /* in/out */
                             unsigned long long seed, unsigned long long step,
                             unsigned long long id_base, long long capacity,
                             void* el_px, void* el_py, void* el_pz, void* el_tau,
                             void* po_px, void* po_py, void* po_pz, void* po_tau,
                             long long* parent, unsigned long long* d_n_out);

/* ---- the whole step of one species in one pass ------------------------------------------
 * qed_step == evolve_optical_depth followed by generate_photons (species = lepton; s1_* = photon
 * buffers, s2_* ignored, may be NULL) or generate_pairs (species = photon; s1_* = electron,
 * s2_* = positron buffers), with identical results, ordering, capacity rule and d_n_out, but the
 * evolve pass also stages a record (momentum, chi^2, index) of every particle that fires (it
 * still has them in registers), so the event pass reads dense records instead of re-scanning tau
 * and gathering scattered parents.  The staging buffer (24 records of 48 B (fp64) or 32 B (fp32)
 * per 128 particles, about 9 bytes per particle in fp64) is owned by the context.  This is the
 * call bench.py times. */
int picsarqed_qed_step(picsarqed_ctx* ctx, int species, int dtype, int tau_dtype, long long n,
                       void* px, void* py, void* pz, /* in/out */
                       const void* ex, const void* ey, const void* ez,
                       const void* bx, const void* by, const void* bz,
                       void* tau, /* in/out */ double dt,
                       unsigned long long seed, unsigned long long step,
                       unsigned long long id_base, long long capacity,
                       void* s1_px, void* s1_py, void* s1_pz, void* s1_tau,
                       void* s2_px, void* s2_py, void* s2_pz, void* s2_tau,
                       long long* parent, unsigned long long* d_n_out);

/* Reads an 8-byte device counter written by the calls above.  Synchronises the stream. */
int picsarqed_read_count(picsarqed_ctx* ctx, const unsigned long long* d_count,
                         unsigned long long* host_out);

/* ---- host-buffer convenience path (used for end-to-end timing) -------------------------
 * One full QED step for one species on HOST arrays: copies the nine particle/field arrays
 * and tau to device staging owned by the context, runs qed_step, copies p, tau and the
 * secondaries back.  The arrays are cut into slabs of whole evolve tiles: slab k+1 is copied in
 * and slab k-1 copied out (three streams, full-duplex PCIe) while slab k is stepped; the slabs
 * are chained through device counters so that the results are bit for bit those of ONE qed_step
 * over the whole arrays (same order of the secondaries, global parent indices, same capacity
 * rule).  All pointers are HOST pointers (pinned memory makes the copies asynchronous and lets
 * them overlap; pageable memory works but serialises).
 * sec[0..3] (leptons: photon px,py,pz,tau) or sec[0..7] (photons: el px,py,pz,tau, po
 * px,py,pz,tau) receive min(*h_n_out, capacity) entries each.  Synchronises. */
int picsarqed_step_host(picsarqed_ctx* ctx, int species, int dtype, int tau_dtype, long long n,
                        void* h_px, void* h_py, void* h_pz,
                        const void* h_ex, const void* h_ey, const void* h_ez,
                        const void* h_bx, const void* h_by, const void* h_bz,
                        void* h_tau, double dt,
                        unsigned long long seed, unsigned long long step,
                        unsigned long long id_base, long long capacity,
                        void* const* h_sec, long long* h_parent, unsigned long long* h_n_out);

/* ---- closed loop in a uniform field ----------------
 * The paper validates the library inside a PIC code on populations in static uniform fields
 * (Ridgers cases (i), (iii)): leptons are pushed, every species takes its QED step, the
 * secondaries join the populations, photons below an energy threshold are dropped at creation,
 * energy spectra are compared (Fig.6).  These calls are the pieces around qed_step that this
 * needs; cascade_step strings them together.  Units as everywhere: p in m_e c, e = E/E_s,
 * b = cB/E_s, dt in seconds. */

/* Boris push of n leptons of charge sign `charge_sign` (-1 electron, +1 positron) by dt in the
 * uniform fields e[3], b[3] (HOST arrays of three doubles): half kick, rotation with
 * t = s b dt/(2 tau_C gamma^-), half kick; du/dt = s (e + u x b/gamma)/tau_C, tau_C = hbar/(m_e c^2)
 * (R19).  px, py, pz: device, in/out.  fp64 arithmetic whatever `dtype`. */
int picsarqed_boris_push_uniform(picsarqed_ctx* ctx, int dtype, long long n, void* px, void* py, void* pz,
                                 int charge_sign, const double* e, const double* b, double dt);

/* ---- chi threshold and classical radiation reaction (R24) -------------------------------
 * "WarpX offers the possibility to select a minimum quantum parameter threshold below which Breit-Wheeler pair production
 * is ignored and photon emission is simulated with a classical model."  set_chi_threshold(chi_min > 0): a particle with
 * chi < chi_min has no event of either kind -- its optical depth is not decremented by chi, evolve_optical_depth,
 * qed_step, step_host or cascade_step (0, the default, switches the threshold off).  classical_loss: one explicit step of
 * the classical model for the leptons below the threshold, d(gamma-1)/dt = -(2/3)(alpha/tau_C) chi^2 (gamma-1)/gamma
 * (the chi -> 0 limit of the mean loss of the Monte Carlo emission), direction kept, momenta rewritten in place; leptons
 * at or above the threshold are not touched; a no-op while the threshold is 0.  Library units only.  cascade_step calls
 * it for both lepton species after the push when the threshold is set. */
int picsarqed_set_chi_threshold(picsarqed_ctx* ctx, double chi_min);
int picsarqed_classical_loss(picsarqed_ctx* ctx, int dtype, long long n, void* px, void* py, void* pz,
                             const void* ex, const void* ey, const void* ez,
                             const void* bx, const void* by, const void* bz, double dt);

/* Ordered, filtering append (R20, R22): of the first m = min(*d_count, m_max) entries
 * of the source arrays s_* (device; *d_count is a device counter such as qed_step's d_n_out),
 * those with sqrt(px^2+py^2+pz^2) >= min_energy (photons below the threshold are
 * discarded right after creation; min_energy = 0 keeps everything) are copied, in order, to
 * d_*[dst_n ...] (device arrays of dst_capacity entries).  *d_new_n (device, 8 bytes) receives
 * dst_n + number kept; entries that would land at or past dst_capacity are not written, so the
 * caller detects overflow by *d_new_n > dst_capacity. */
int picsarqed_append_secondaries(picsarqed_ctx* ctx, int dtype, int tau_dtype, long long m_max,
                                 const void* s_px, const void* s_py, const void* s_pz, const void* s_tau,
                                 const unsigned long long* d_count, double min_energy,
                                 void* d_px, void* d_py, void* d_pz, void* d_tau,
                                 long long dst_n, long long dst_capacity, unsigned long long* d_new_n);

/* Energy spectrum (Fig.6; R23): adds to hist[nbins] (device, 64-bit counters, NOT
 * zeroed here) the number of particles per logarithmic bin of [e_min, e_max) of the kinetic energy
 * gamma - 1 (leptons) or gamma_gamma = |p| (photons); bin = floor((ln E - ln e_min) nbins /
 * (ln e_max - ln e_min)) in fp64.  Dead entries (p = 0) and energies outside the range are not
 * counted.  1 <= nbins <= 8192. */
int picsarqed_energy_spectrum(picsarqed_ctx* ctx, int species, int dtype, long long n,
                              const void* px, const void* py, const void* pz,
                              double e_min, double e_max, int nbins, unsigned long long* hist);

/* One species of the closed loop: device structure of arrays with room for `capacity` entries, the
 * first n in use.  Positions never change (a photon that decayed stays as p = 0, tau = +inf), so the
 * Philox id of a particle is id_base + position for its lifetime (R21). */
typedef struct picsarqed_species_arrays {
    void *px, *py, *pz, *tau;
    long long n;        /* in/out */
    long long capacity;
    unsigned long long id_base;
} picsarqed_species_arrays;

/* One time step of the closed loop in the order of DESIGN.md R20: push electrons (s = -1) and
 * positrons (+1); qed_step of electrons, positrons, photons in the uniform field (each on the
 * entries that existed when the step began); append the photons of the electrons, then those of
 * the positrons (min_energy = photon_min_energy), and the pairs.  Updates n of the three species
 * (one 24-byte device-to-host read per step) and writes the event counts (electrons, positrons,
 * photons) to h_events[3] if it is not NULL.  Scratch (constant field arrays, secondary buffers) is
 * owned by the context.  PICSARQED_ERR_INVALID if a species would exceed its capacity (its n is
 * then clipped to the capacity and the entries that did not fit are lost).  * The Philox counter distinguishes leptons from photons only, so electrons and positrons must own disjoint id ranges
 * [id_base, id_base + capacity) (e.g. 0 and 2^40; R21): cascade_step returns PICSARQED_ERR_INVALID otherwise.
 */
int picsarqed_cascade_step(picsarqed_ctx* ctx, int dtype, int tau_dtype,
                           picsarqed_species_arrays* electrons, picsarqed_species_arrays* positrons,
                           picsarqed_species_arrays* photons, const double* e, const double* b, double dt,
                           unsigned long long seed, unsigned long long step, double photon_min_energy,
                           int push, unsigned long long* h_events);

/* ---- the table functions per value (Figs.2-5) ---------------------
 * What the hot path evaluates, exposed for single values so that table accuracy can be studied
 * (error against table size) and so that a caller can sample
 * outside a particle loop.  chi, r, out: device arrays of n reals of type `dtype`.
 *
 * table_function: kind 0: out[i] = G(chi[i]) by eq.27 (first/last value outside the table);
 * kind 1: out[i] = T(chi[i]) by eq.23 inside the table, the Erber form outside.
 * The kernel runs the evolve pass's own routine on a synthetic particle of that chi. */
int picsarqed_table_function(picsarqed_ctx* ctx, int kind, int dtype, long long n, const void* chi, void* out);

/* sample_xi: kind 0: xi = chi_gamma/chi of the emitted photon by eqs.28-30 from r[i] in (0,1);
 * kind 1: xi = chi_-/chi_gamma of the electron of the pair by eqs.24-26, with the reflection
 * r -> 1 - r, xi -> 1 - xi for r > 1/2.  The routines are those of the event pass. */
int picsarqed_sample_xi(picsarqed_ctx* ctx, int kind, int dtype, long long n, const void* chi, const void* r,
                        void* xi_out);

#ifdef __cplusplus
}
#endif
#endif /* PICSARQED_H */
