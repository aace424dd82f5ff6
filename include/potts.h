/*
 * potts.h -- C-ABI boundary of the B200-native checkerboard Metropolis sweep of the 2D q-state
 * Potts model (arXiv 1101.0876; citations are PAPER.md:<line>, section/equation).
 *
 * The library implements, entirely in hand-written CUDA for sm_100a, the one data-parallel hot
 * path of the paper: the red/black single-spin-flip Metropolis sweep (sec. 3,
 * :141 sec. 3.1) of  H = -J sum_<ij> delta(s_i,s_j)  (Eq. 1) on an L x L periodic
 * square lattice, and the per-sweep energy and q-state occupancy reduction (PAPER.md:175
 * sec. 3.4) that feeds the metastability analysis (sec. 6).
 *
 * Conventions
 *   - Every function returns a POTTS_* code and never throws.  On any error the out-parameters
 *     are left untouched and potts_last_error() describes the failure (thread-local string).
 *   - "host" / "device" is stated for every pointer.  Host buffers are caller-owned; the handle
 *     owns its device memory until potts_destroy (or borrows the caller's workspace, see
 *     potts_create_ex).
 *   - All device work is enqueued on the handle's CUDA stream (default: the legacy default
 *     stream; the Python binding installs torch's current stream).  potts_sweep may return
 *     before the GPU finishes; every function that fills a host buffer synchronises the stream.
 *   - One handle = one lattice.  Handles are independent.  A handle is not thread-safe.
 *   - There is no CPU fallback: without a usable CUDA device every call fails with
 *     POTTS_ERR_CUDA.
 *
 * The simulated chain (what the bits are), see DESIGN.md section 3 for the readings:
 *   spins s in {0..q-1}; J = k_B = 1; sweep t = all sites with (i+j) even, then all with (i+j)
 *   odd; per site (w0,w1,..) = Philox4x32-10(counter (j, i, t, colour), key seed); proposal
 *   s' = floor(w0 q / 2^32); d = n_old - n_new over the 4 neighbours; accept iff d <= 0 or
 *   w1 < floor(2^32 exp(-d/T)).  No floating point is used on the device.
 */
#ifndef POTTS_B200_H
#define POTTS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct potts_s potts_t; /* opaque */

enum {
    POTTS_OK = 0,
    POTTS_ERR_ARG = 1,         /* null pointer, L < 2 or odd, q outside [2,256], T not finite or <= 0,
                                  nsweeps < 0, every < 1 or not dividing nsweeps, bad init/layout,
                                  spin value >= q in an upload, sweep counter would pass 2^32 - 1 */
    POTTS_ERR_UNSUPPORTED = 2, /* L not a multiple of 32 (vector width of the kernels; 64 for the packed
                                  layout), q > 32 with the packed layout, or a forced launch variant that
                                  cannot hold this lattice */
    POTTS_ERR_NOMEM = 3,       /* device or host allocation failed / workspace too small */
    POTTS_ERR_CUDA = 4         /* CUDA runtime error (no device, launch failure, ...) */
};

enum { POTTS_INIT_ORDERED = 0 /* all s = 0 */, POTTS_INIT_RANDOM = 1 /* uniform {0..q-1} from seed */ };

enum {
    POTTS_LAYOUT_U8 = 0,    /* one byte per spin, split by colour */
    POTTS_LAYOUT_PACKED = 1 /* sub-byte, q <= 32, L % 64 == 0: 4 bits per spin (nibble plane) for q <= 16,
                               5 bits (nibble plane + high-bit plane) for 16 < q <= 32; DESIGN.md section 5.
                               Results are bit-identical to U8 */
};

/* ---- lifetime ------------------------------------------------------------------------------
 * potts_create: allocate an L x L lattice with q states (byte spins, q <= 256,
 * PAPER.md:161), Philox key `seed`, start state `init` (ordered / random), sweep
 * counter t = 0, layout U8, on the current CUDA device.  *out (host) receives the handle. */
int potts_create(potts_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init);

/* potts_create_ex: as potts_create, with a layout and optionally caller-provided device memory
 * and stream.  If dev_workspace (device) is non-null it must hold at least
 * potts_workspace_bytes(...) bytes, be 256-byte aligned, and outlive the handle (the handle
 * does not free it); if null the library allocates.  cuda_stream is a cudaStream_t (may be
 * null = legacy default stream). */
int potts_create_ex(potts_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, int32_t layout,
                    void *dev_workspace, size_t workspace_bytes, void *cuda_stream);

/* Bytes of device memory a handle needs (spin planes + accumulators).  *bytes is host. */
int potts_workspace_bytes(int32_t L, int32_t q, int32_t layout, size_t *bytes);

/* Install the cudaStream_t all later work of this handle is enqueued on. */
int potts_set_stream(potts_t *h, void *cuda_stream);

void potts_destroy(potts_t *h);

/* ---- the hot path --------------------------------------------------------------------------
 * potts_sweep: nsweeps checkerboard Metropolis sweeps at temperature T (PAPER.md:94, :141,
 * :145).  The four acceptance thresholds floor(2^32 exp(-d/T)) are built on the host in double
 * at every call.  Enqueues and returns; advances the sweep counter by nsweeps.
 * potts_sweep(h,T,a); potts_sweep(h,T,b) is the same chain as potts_sweep(h,T,a+b). */
int potts_sweep(potts_t *h, double T, int64_t nsweeps);

/* potts_sweep_measured: as potts_sweep, and after every `every`-th sweep of this call record
 * the energy E (Eq. 1, int64) and, if hist_series is non-null, the occupancies N_0..N_{q-1}
 * ("one measure each delta-t steps").  E_series (host) has
 * nsweeps/every entries, hist_series (host) nsweeps/every rows of q.  Synchronises. */
int potts_sweep_measured(potts_t *h, double T, int64_t nsweeps, int64_t every,
                         int64_t *E_series, int64_t *hist_series);

/* potts_sweep_delta: as potts_sweep, and for every sweep of this call record the energy CHANGE of that sweep
 * accumulated on the fly from the accepted moves, dE = sum of d = n_old - n_new over accepted updates of both
 * colours, without recounting the energy over the lattice -- the "parallel accumulation of local
 * energy changes on-the-fly" that PAPER.md:361-363 proposes for reweighting / histogram techniques.  By Eq. 1
 * E(after sweep n) = E(before) + dE_series[n]; the tests check exactly that against the oracle's
 * recounted energies.  dE_series: caller-owned HOST buffer of nsweeps int64.  Both layouts; always one launch
 * per half-sweep (k_half_sweep_delta_u8, or k_half_sweep_packed in its delta form).  Synchronises; dE_series is
 * untouched on error. */
int potts_sweep_delta(potts_t *h, double T, int64_t nsweeps, int64_t *dE_series);

/* Same, with E_series / hist_series in DEVICE memory; enqueues and returns without a sync. */
int potts_sweep_measured_dev(potts_t *h, double T, int64_t nsweeps, int64_t every,
                             int64_t *E_series_dev, int64_t *hist_series_dev);

/* potts_ladder: the paper's simulation protocol (sec. 3: "fix T, run t_tran sweeps, then t_max sweeps
 * with one measure each delta-t steps, keep the last configuration for the next T").  For each temperature T[k]
 * (host, nT entries, in the order given: ascending = heating, descending = cooling): t_tran unmeasured sweeps,
 * then t_max sweeps recording E and, if hist_series is non-null, N_0..N_{q-1} after every dt-th.  Configuration
 * and sweep counter carry over.  E_series (host): nT rows of t_max/dt entries; hist_series (host): nT * t_max/dt
 * rows of q.  Everything is enqueued at once; one synchronisation at the end.  Same chain as the equivalent
 * sequence of potts_sweep / potts_sweep_measured calls. */
int potts_ladder(potts_t *h, const double *T, int32_t nT, int64_t t_tran, int64_t t_max, int64_t dt,
                 int64_t *E_series, int64_t *hist_series);

/* ---- replica batch (the paper averages over samples and scans temperatures) --------
 * n independent lattices of the same (L, q), lattice r with Philox key seeds[r], all advanced by one kernel launch
 * per call: CTA r keeps lattice r in its shared memory (U8 layout, L % 32 == 0, 2 (L+2) L/2 bytes must fit one CTA:
 * L <= 416).  Lattice r of a batch follows exactly the chain of a single handle created with (L, q, seeds[r], init).
 * seeds, T: host arrays of n entries.  dev_workspace: device memory of potts_batch_workspace_bytes() bytes, 256-byte
 * aligned, or null (the library allocates).  */
typedef struct potts_batch_s potts_batch_t;
int potts_batch_workspace_bytes(int32_t n, int32_t L, int32_t q, size_t *bytes);
int potts_batch_create(potts_batch_t **out, int32_t n, int32_t L, int32_t q, const uint64_t *seeds, int32_t init,
                       void *dev_workspace, size_t workspace_bytes, void *cuda_stream);
void potts_batch_destroy(potts_batch_t *b);
/* nsweeps sweeps of every lattice, lattice r at temperature T[r].  If E_series / hist_series (host; n rows of
 * nsweeps/every entries / of nsweeps/every x q) are non-null, record after every `every`-th sweep; with both null
 * `every` is ignored.  Synchronises. */
int potts_batch_sweep_measured(potts_batch_t *b, const double *T, int64_t nsweeps, int64_t every,
                               int64_t *E_series, int64_t *hist_series);
/* The same with DEVICE series (int64, n rows of nsweeps/every entries / x q; zeroed by the call), no synchronisation. */
int potts_batch_sweep_measured_dev(potts_batch_t *b, const double *T, int64_t nsweeps, int64_t every,
                                   int64_t *E_series_dev, int64_t *hist_series_dev);
/* potts_batch_sweep_delta: nsweeps sweeps of every lattice; dE_series (host, n rows of nsweeps int64) receives for
 * every lattice and sweep the energy change summed over the accepted moves, as potts_sweep_delta. */
int potts_batch_sweep_delta(potts_batch_t *b, const double *T, int64_t nsweeps, int64_t *dE_series);
/* potts_batch_ladder: the temperature-ladder protocol for every lattice of the batch at once.
 * T: host, n rows of nT temperatures (lattice r runs T[r*nT + k], k = 0..nT-1, state carried over); per temperature
 * t_tran unmeasured sweeps, then t_max sweeps sampled every dt.  E_series / hist_series (host, may be null): n rows of
 * nT * t_max/dt samples (x q).  Lattice r follows exactly potts_ladder of a single handle with (seeds[r], T row r). */
int potts_batch_ladder(potts_batch_t *b, const double *T, int32_t nT, int64_t t_tran, int64_t t_max, int64_t dt,
                       int64_t *E_series, int64_t *hist_series);
int potts_batch_download(potts_batch_t *b, int32_t r, uint8_t *spins); /* lattice r, host, L*L row-major */
int potts_batch_sweep_count(potts_batch_t *b, uint64_t *t);
int potts_batch_launch_count(potts_batch_t *b, uint64_t *n);

/* ---- measurements (sec. 3.4) ---------------------------------------------------
 * potts_energy: E = -(number of satisfied nearest-neighbour bonds), range [-2 L^2, 0].  *E host. */
int potts_energy(potts_t *h, int64_t *E);

/* potts_histogram: counts[k] = #{sites with s = k}, k = 0..q-1 (host, q entries, caller-owned). */
int potts_histogram(potts_t *h, int64_t *counts);

/* ---- state transfer --------------------------------------------------------------------------
 * potts_download: spins (host, L*L bytes, row-major s[i*L + j]) <- current configuration.
 * Together with potts_sweep_count this is a complete checkpoint (the RNG is stateless). */
int potts_download(potts_t *h, uint8_t *spins);

/* potts_upload: replace the configuration (host, L*L bytes, every value < q). */
int potts_upload(potts_t *h, const uint8_t *spins);

int potts_sweep_count(potts_t *h, uint64_t *t);
int potts_set_sweep_count(potts_t *h, uint64_t t); /* checkpoint restore; t < 2^32 */

/* ---- host-side derived observables in double (PAPER.md:73 Eq. 7, :209 Eq. 9) ----------------
 * From an energy series of n samples of a lattice with N = L^2 sites at temperature T:
 *   *mean_e = <E>/N,  *cv = (<E^2> - <E>^2)/(N T^2),  *binder = 1 - <E^4>/(3 <E^2>^2).
 * Sums of E and E^2 are exact (128-bit integers), E^4 is summed compensated in long double.
 * All pointers host; any out-pointer may be null. */
int potts_observables(const int64_t *E_series, int64_t n, int64_t N, double T,
                      double *mean_e, double *cv, double *binder);

/* *m = (q N_max/N - 1)/(q - 1) from a histogram (host, q entries). */
int potts_magnetisation(const int64_t *counts, int32_t q, double *m);

/* potts_susceptibility (Eq. 11, with m of PAPER.md:73 Eq. 7): from a series of n histograms
 * (host, n rows of q int64 counts, every row summing to the same N > 0)
 *   *mean_m = <m>,  *mean_m2 = <m^2>,  *chi = N/T (<m^2> - <m>^2).
 * With a_k = q Nmax_k - N (an integer) m_k = a_k / ((q-1) N); sum a_k and sum a_k^2 are formed exactly in 128-bit
 * integers, and so is n sum a^2 - (sum a)^2 (long double beyond 2^126), then one conversion: robust against the
 * cancellation in the variance.  Any out-pointer may be null.  POTTS_ERR_ARG: null series, n < 1, q outside
 * [2, 256], T not finite or <= 0, a negative count, rows with different or zero sums. */
int potts_susceptibility(const int64_t *hist_series, int64_t n, int32_t q, double T,
                         double *mean_m, double *mean_m2, double *chi);

/* ---- random-stream definition ---------------------------------------------------------------------------------
 * potts_set_stream_spec: 1 (default) = one Philox4x32-10 block per site and half-sweep, words (w0, w1), as in the
 * header comment; 2 = "stream-spec v2" (reading S15): the same-colour sites of a row are numbered k = j>>1,
 * sites 2m and 2m+1 share the block of counter (j of site 2m, i, t, colour), site 2m takes (w0, w1), site 2m+1
 * (w2, w3).  This is NOT a launch option: it selects another Markov chain (same rules, same stationary distribution,
 * other random numbers, half the random-number work).  Takes effect for all later sweeps of the handle. */
int potts_set_stream_spec(potts_t *h, int32_t spec);
int potts_get_stream_spec(potts_t *h, int32_t *spec);
int potts_batch_set_stream_spec(potts_batch_t *b, int32_t spec);

/* ---- introspection / tuning -------------------------------------------------------------------
 * potts_launch_count: kernels launched by this handle since creation (bench.py's gpu_launches). */
int potts_launch_count(potts_t *h, uint64_t *n);

/* potts_set_option: tuning knobs that change HOW the sweep is launched, never WHAT it computes
 * (tests assert bit-identity across them).  Unknown key -> POTTS_ERR_ARG.  Keys:
 *   "variant"          0 = automatic, 1 = streaming (one kernel launch per half-sweep, planes read through
 *                      L2/HBM), 2 = resident (one persistent cooperative launch per call, lattice in shared
 *                      memory; U8 layout, L <= 4096; POTTS_ERR_UNSUPPORTED from the sweep call otherwise)
 *                      3 = cluster (one thread-block cluster of up to 16 CTAs, boundary rows through distributed
 *                      shared memory; the automatic choice for L <= 288)
 *   "cluster_ctas"     0 = automatic, else the cluster size (1..16); "cluster_active" (read-only) = the cluster
 *                      size the next sweep call would use, 0 if it would not use the cluster kernel
 *   "resident_ctas"    0 = automatic, else the number of CTAs the resident kernel splits the rows over
 *   "resident_rows"    0 = automatic, else at most this many thread rows in a resident block
 *   "resident_words"   0 = automatic, 1 / 2 = 4-site words a resident thread updates per row visit
 *   "resident_active"  read-only: CTAs the next sweep call would run resident on (0 = streaming) */
int potts_set_option(potts_t *h, const char *key, int64_t value);
int potts_get_option(potts_t *h, const char *key, int64_t *value);

/* Description of the last failure on this thread ("" if none). */
const char *potts_last_error(void);

/* Library version string, e.g. "potts-b200 0.1 (sm_100a)". */
const char *potts_version(void);

/* ---- one lattice split into row strips over several GPUs -------------------------------------------------
 * A strip handle holds rows [row0, row0 + rows) of the L x L lattice (U8 layout, both ends multiples of 32) plus one
 * halo row above and one below per colour plane.  Because the random words are a pure function of the GLOBAL site
 * (R3) the strips together follow exactly the chain of one potts_create handle, whatever their number.  The caller
 * drives the sweep: for colour 0 then 1: potts_strip_half_sweep on every strip, then copy each strip's first / last
 * row of the plane just written (potts_strip_rows: device pointers, row_bytes = L/2) into the halo_below / halo_above
 * of the strip above / below it (periodic; device-to-device or NCCL send/recv); then potts_strip_advance.  Before the
 * first half-sweep the halos of BOTH planes must be filled the same way.  E_dev (colour 1 only) / hist_dev: device
 * int64 accumulators (1 / q entries, zeroed by the caller) that receive this strip's part of the energy / histogram
 * of the sites just written, or null.  potts_energy, potts_histogram (partial sums over the strip; the halos of plane 0
 * must be current), potts_download / potts_upload (rows x L bytes) work on strip handles; potts_sweep* do not
 * (POTTS_ERR_UNSUPPORTED).  paper_1101_0876_b200/strips.py drives strips over torch.distributed. */
int potts_create_strip(potts_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, int32_t row0, int32_t rows,
                       void *cuda_stream);
int potts_strip_half_sweep(potts_t *h, double T, int32_t colour, int64_t *E_dev, int64_t *hist_dev);
int potts_strip_advance(potts_t *h);
int potts_strip_rows(potts_t *h, int32_t colour, void **first_row, void **last_row, void **halo_above, void **halo_below,
                     size_t *row_bytes);

/* ---- 3D generalisation (sec. 7: "For the generalization to the 3D case, the checkerboard scheme defining
 * two independent sub-networks persists, however the cell-packing scheme should be updated") -----------------------
 * The same Metropolis chain on an L x L x L periodic simple-cubic lattice with 6 nearest neighbours (DESIGN.md reading
 * S16): E = -sum over sites of [delta(s, s_{x+1}) + delta(s, s_{y+1}) + delta(s, s_{z+1})] in [-3 L^3, 0]; sweep = all
 * sites with (x+y+z) even, then all with (x+y+z) odd; random words Philox4x32-10(counter = (x, y, t, colour + 4 z),
 * key = seed); proposal floor(w0 q / 2^32); accept iff d <= 0 or w1 < floor(2^32 exp(-d/T)), d = n_old - n_new in
 * -6..6; random start from counter (x, y, 0, 2 + 4 z).  Spins cross the boundary as s[(z L + y) L + x] (host, L^3
 * bytes).  L even, L % 32 == 0 (POTTS_ERR_UNSUPPORTED otherwise), L <= 2048; U8 layout only.  cuda_stream: the stream
 * every call of the handle uses (null = default stream).  Conventions as for potts_t: return codes, potts_last_error(),
 * out-parameters untouched on error, potts3_sweep may return before the GPU finishes, the others synchronise.
 * E_series / hist_series of potts3_sweep_measured: host, nsweeps/every entries (x q), either may be null. */
typedef struct potts3_s potts3_t;
int  potts3_create(potts3_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, void *cuda_stream);
void potts3_destroy(potts3_t *h);
int  potts3_sweep(potts3_t *h, double T, int64_t nsweeps);
int  potts3_sweep_measured(potts3_t *h, double T, int64_t nsweeps, int64_t every, int64_t *E_series, int64_t *hist_series);
int  potts3_energy(potts3_t *h, int64_t *E);
int  potts3_histogram(potts3_t *h, int64_t *counts);
int  potts3_download(potts3_t *h, uint8_t *spins);
int  potts3_upload(potts3_t *h, const uint8_t *spins);
int  potts3_sweep_count(potts3_t *h, uint64_t *t);
int  potts3_set_sweep_count(potts3_t *h, uint64_t t);
int  potts3_launch_count(potts3_t *h, uint64_t *n);
/* potts3_set_option: launch knobs of the 3D half-sweep that never change WHAT it computes (tests assert bit-identity
 * across them).  Unknown key or bad value -> POTTS_ERR_ARG.  Keys:
 *   "stream_words"  0 = automatic (4; the one-chunk-per-thread kernel where a quarter of the lanes would idle, L = 3 2^k),
 *                   1 / 2 / 4 = 4-site words a lane of the row-walking kernel k_sweep3_rows_u8 updates per row visit,
 *                   -1 = the one-chunk-per-thread kernel k_sweep3_u8
 *   "stream_rows"   0 = automatic (16, halved while a launch would have fewer than 1024 tiles), else rows a lane walks
 *                   per tile (2, 4, 8, 16 or 32) */
int  potts3_set_option(potts3_t *h, const char *key, int64_t value);

/* ---- first AND second neighbour interactions (sec. 7: "For the 2D case with first and second neighbors
 * interactions, there are nine independent sub-networks to update instead of two") --------------------------------
 * The same Metropolis chain on the L x L periodic square lattice where every site interacts with its 4 first and its 4
 * second (diagonal) neighbours, equal coupling J = 1 (reading S17):
 * E = -sum over sites of [d(s, s_{i,j+1}) + d(s, s_{i+1,j}) + d(s, s_{i+1,j+1}) + d(s, s_{i+1,j-1})] in [-4 L^2, 0];
 * sweep = the nine sub-networks c = 3 (i mod 3) + (j mod 3), c = 0..8 in this order; random words
 * Philox4x32-10(counter = (j, i, t, 16 + c), key = seed); d = n_old - n_new in -8..8, thresholds floor(2^32 exp(-d/T)),
 * d = 1..8; start states as potts_create (the random start is the same configuration).  Spins cross the boundary
 * row-major s[i L + j] (host).  L a multiple of 3 (POTTS_ERR_ARG otherwise) and of 12 (POTTS_ERR_UNSUPPORTED otherwise).
 * Conventions as for potts3_*. */
typedef struct potts8_s potts8_t;
int  potts8_create(potts8_t **out, int32_t L, int32_t q, uint64_t seed, int32_t init, void *cuda_stream);
void potts8_destroy(potts8_t *h);
int  potts8_sweep(potts8_t *h, double T, int64_t nsweeps);
int  potts8_sweep_measured(potts8_t *h, double T, int64_t nsweeps, int64_t every, int64_t *E_series, int64_t *hist_series);
int  potts8_energy(potts8_t *h, int64_t *E);
int  potts8_histogram(potts8_t *h, int64_t *counts);
int  potts8_download(potts8_t *h, uint8_t *spins);
int  potts8_upload(potts8_t *h, const uint8_t *spins);
int  potts8_sweep_count(potts8_t *h, uint64_t *t);
int  potts8_set_sweep_count(potts8_t *h, uint64_t t);
int  potts8_launch_count(potts8_t *h, uint64_t *n);
/* potts8_set_option: launch knobs that never change WHAT is computed.  Unknown key or bad value -> POTTS_ERR_ARG.  Keys:
 *   "stream_words"  0 = automatic (the row-walking kernel k_sweep8_rows_u8, 16 sites per lane and row visit, for
 *                   L >= 3072 with L % 48 == 0; else the one-word-per-thread kernel k_sweep8_u8), 4 = k_sweep8_rows_u8
 *                   wherever L % 48 == 0 and L < 65536, -1 = k_sweep8_u8
 *   "stream_rows"   0 = automatic (16, halved while a launch would have fewer than 1024 tiles), else rows a lane walks
 *                   per tile (1, 2, 4, 8 or 16) */
int  potts8_set_option(potts8_t *h, const char *key, int64_t value);

/* ---- no-allocation entry point ------------------------------------------------------------------------------------
 * potts_measure_noalloc: energy (R1: E = -(number of satisfied bonds), Eq. 1) and q-bin histogram (R8,
 * PAPER.md:175) of a lattice the CALLER holds on the device, for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it).  The same kernel as potts_energy / potts_histogram
 * (k_measure_u8), with its colour planes and accumulators in a file-scope device array of fixed size instead of a
 * handle's cudaMalloc'ed workspace: the call allocates and frees nothing, needs no handle, and every GPU that loads the
 * library holds that array (POTTS_NOALLOC_MAX_L^2 + 4096 bytes = 4 MiB + 4 KiB) until the process exits.
 *   spins_dev  DEVICE pointer, L*L bytes, row-major s[i*L + j] in 0..q-1, 8-byte aligned; read only
 *   L, q       L even, L % 32 == 0 (POTTS_ERR_UNSUPPORTED otherwise), L <= POTTS_NOALLOC_MAX_L (POTTS_ERR_UNSUPPORTED
 *              beyond: use a potts_t handle); 2 <= q <= 256
 *   E_dev      DEVICE pointer to one int64, or null;  hist_dev  DEVICE pointer to q int64, or null (not both null);
 *              caller-owned, written by the call.  A spin value >= q cannot be reported through the return code
 *              without a synchronisation: it sets *E_dev = INT64_MIN and every hist_dev[k] = -1 instead.
 *   cuda_stream  the stream the work is enqueued on (null = default stream); the device of the pointers must be current.
 * The call returns once the work is enqueued (no synchronisation); results are valid when the stream reaches that point.
 * The first call on a device resolves the array's address (cudaGetSymbolAddress; this may load the module): a caller
 * that captures graphs makes one call outside capture first.  ALL calls share the one array: it is cleared where needed
 * at the start of each call, and calls that overlap on the GPU (different streams without ordering, several host
 * threads) race on it -- the caller serialises them.  Argument errors are returned before any CUDA call. */
#define POTTS_NOALLOC_MAX_L 2048
int  potts_measure_noalloc(const uint8_t *spins_dev, int32_t L, int32_t q, int64_t *E_dev, int64_t *hist_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* POTTS_B200_H */
