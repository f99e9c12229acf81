/* include/mpr.h -- C ABI of libmpr.so: the conditional hybrid Monte-Carlo hot path of the
 * modified planar rotator (MPR) prediction method, hand-written CUDA for sm_100a (B200).
 *
 * What the library computes (arxiv/paper_1910_08448; PAPER.md:N = line N of the paper text,
 * DESIGN.md section 3 lists the readings R1..R17 where the paper is silent):
 *   - H = -J sum_<ij> cos[q (phi_i - phi_j)], phi in [0, 2pi], q = 1/2, J = 1
 *                                                        PAPER.md:27-29 (Eq. 2)
 *   - "maps the measured data onto spins"                PAPER.md:13 (sec. 1), R1
 *   - "the temperature ... needs to be inferred from the incomplete data"
 *                                                        PAPER.md:31 (sec. 2), R6
 *   - "a conditional Monte Carlo simulation, in which only the spins at the prediction
 *     locations are allowed to change their states ... hybrid algorithm"
 *                                                        PAPER.md:31 (sec. 2), R4/R5/R7
 *   - "averaging over multiple configurations in equilibrium" -> prediction
 *                                                        PAPER.md:31 (sec. 2), R15
 *   - specific energy e = <H>/L^2                        PAPER.md:35 (sec. 2), R3
 *   - precision settings (spins, energy, functions)      PAPER.md:35 (sec. 2), R12/R13
 *
 * Conventions for every call
 *   - Pointers named d_* are DEVICE pointers, h_* / plain scalars are HOST memory.
 *   - Grids are row-major, site index s = y*L + x, 0 <= x,y < L.
 *   - Ownership: the caller owns every buffer (inputs, outputs, workspace); the library
 *     allocates no device memory (its only device storage of its own is the fixed 49 KB scratch array of
 *     mpr_sample_energy_static) and creates no stream.  It borrows d_values, d_mask and
 *     the workspace for the life of the context and never writes d_values / d_mask.
 *   - Errors: every call returns 0 (MPR_OK) or a negative mpr_status.  Nothing is thrown,
 *     printed or aborted.  mpr_last_error() gives a text for the last failure of a context.
 *   - Ordering: all device work is enqueued on the context's stream.  Calls that return
 *     host scalars (create, set_workspace, estimate_temperature, run, get_counters, get_energy_series,
 *     get_launch_stats) synchronise that stream before returning; the others are asynchronous.
 *   - Determinism: for fixed (inputs, seed, mode, T) the spin state after any number of
 *     sweeps is bit-identical for every kernel path, tile size and fused depth, and for any cut of the grid into
 *     slabs (mpr_set_slab).
 *   - There is no CPU fallback: without a CUDA device every compute call returns MPR_ERR_CUDA.
 */
#ifndef MPR_H_
#define MPR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mpr_ctx mpr_ctx; /* opaque, host-side */

typedef enum {
  MPR_OK = 0,
  MPR_ERR_INVALID_ARG = -1,      /* L < 2, null pointer, bad mode, negative count, T <= 0   */
  MPR_ERR_NO_MEASURED = -2,      /* no measured site, or no measured nearest-neighbour pair */
  MPR_ERR_DEGENERATE_RANGE = -3, /* z_max == z_min over the measured sample                 */
  MPR_ERR_NONFINITE = -4,        /* NaN/Inf at a measured site                              */
  MPR_ERR_WORKSPACE = -5,        /* workspace null, misaligned (256 B) or too small         */
  MPR_ERR_NOT_READY = -6,        /* run before a temperature was set or estimated           */
  MPR_ERR_NO_ROOT = -7,          /* e_sample outside the reachable e(T) range, R6           */
  MPR_ERR_CUDA = -8              /* a CUDA call failed (no device, launch error, ...)       */
} mpr_status;

/* Precision modes (triple = spins / energy / functions; R12):
 *   MPR_DP            DDD  double storage, double arithmetic and functions
 *   MPR_SP            SSD  float storage of the spins, double arithmetic and functions
 *   MPR_SP_PRECISE    float storage and arithmetic, sinf/cosf/expf (not in the paper)
 *   MPR_SP_INTRINSIC  SSS  float storage and arithmetic, __sinf/__cosf/__expf
 * Energy sums are accumulated in double in every mode (R13) unless X_E = S is asked for (below).
 *   MPR_DS_INTRINSIC  D.S  double storage of the spins, float arithmetic with the intrinsics
 *   MPR_HP            half-precision storage of the spins (two fp16 per spin, 4 bytes), float arithmetic with the
 *                     intrinsics -- the paper's outlook.  The stored vectors carry a 5e-4 relative rounding,
 *                     which shows in e; predictions meet the same 1 % gate as the float modes.
 * The paper's eight settings (X_S X_E X_F) = (spin storage, energy variable, functions), each D or S, are
 * mpr_set_precision_triple("DDD" ... "SSS"): X_S, X_F select the mode (DD -> MPR_DP, SD -> MPR_SP,
 * DS -> MPR_DS_INTRINSIC, SS -> MPR_SP_INTRINSIC), X_E = S makes the energy variable a float
 * (mpr_set_energy_precision): every bond term and every partial sum of the energy reduction is then rounded to float. */
typedef enum { MPR_DP = 0, MPR_SP = 1, MPR_SP_PRECISE = 2, MPR_SP_INTRINSIC = 3, MPR_DS_INTRINSIC = 4,
               MPR_HP = 5 } mpr_precision;

/* Kernel paths.  All give bit-identical spin states (determinism contract).
 *   MPR_PATH_AUTO    (default) the path measured fastest for the mode, grid size and schedule: STRIP for
 *                    MPR_SP_INTRINSIC at L >= 4096 and for the site-fused schedule, TILED otherwise.
 *   MPR_PATH_STRIP   one launch per k <= 2 hybrid sweeps: every warp streams a column strip of
 *                    the grid through a private shared-memory ring fed by TMA and runs the colour
 *                    passes as a software pipeline down the rows (no barriers, no redundant rows).
 *   MPR_PATH_TILED   one launch per hybrid sweep group: TMA stages a tile + halo of both colour
 *                    planes in shared memory, all 4*k colour passes of k sweeps run there.
 *   MPR_PATH_PLAIN   one launch per colour pass on the global colour planes (reference path
 *                    for the self-consistency tests; also used for odd R8 quench passes).
 *   MPR_PATH_LIST    one launch per colour pass over the COMPACTED list of the prediction sites of that
 *                    colour (built at set-up): work proportional to the number of prediction sites,
 *                    neighbour reads are gathers.  For small masked fractions.               */
typedef enum { MPR_PATH_TILED = 0, MPR_PATH_PLAIN = 1, MPR_PATH_STRIP = 2, MPR_PATH_AUTO = 3,
               MPR_PATH_LIST = 4 } mpr_path;

/* Order of the colour passes inside one hybrid sweep ("hybrid algorithm" -- the paper
 * leaves the order to its ref. [5]; both orders leave the conditional Boltzmann density invariant):
 *   MPR_SCHEDULE_R4          (default, R4)  Metropolis colour 0, colour 1, over-relaxation colour 0, 1
 *   MPR_SCHEDULE_SITE_FUSED  (R4b)  per colour, every site gets its Metropolis move and at once its
 *                            over-relaxation move (both read only the other colour): colour 0, colour 1.
 * Same random numbers per (site, sweep); a different, equally valid Markov chain.  Runs on the STRIP
 * and PLAIN paths.                                                                          */
typedef enum { MPR_SCHEDULE_R4 = 0, MPR_SCHEDULE_SITE_FUSED = 1 } mpr_schedule;

/* Bytes of workspace mpr_create needs for an L x L grid (any mode).  HOST out pointer.     */
int mpr_workspace_bytes(int L, size_t* bytes);

/* The paper's problem statement: an L x L grid, values at the measured
 * sites, a set of prediction sites.
 *   d_values  f64[L*L]  value at measured sites; never read where d_mask == 1 (may be NaN)
 *   d_mask    u8 [L*L]  1 = prediction ("free") site, 0 = measured site
 *   d_workspace         >= mpr_workspace_bytes(L) bytes, 256-byte aligned
 *   cuda_stream         a cudaStream_t (0 = default stream)
 * Does R1 (z_min, z_max over the measured sample, phi = 2pi (z - z_min)/(z_max - z_min)),
 * the sample energy of R6 (e_s over measured nearest-neighbour pairs), packs the mask into
 * per-colour bitmaps, selects MPR_DP, seed 0, and resets the chain (R8).  "Resets the chain"
 * here and in the setters below means: the chain is marked for re-initialisation (uniform
 * spins + quench passes, trial 0), which runs once, on the stream, when the chain is next
 * used (run, sweep, pass, get/set_state, energy, counters) -- create + set_precision +
 * set_seed costs one initialisation, not three.
 * Fails with INVALID_ARG, WORKSPACE, NO_MEASURED, DEGENERATE_RANGE, NONFINITE or CUDA;
 * *out is null on failure.
 * Two-step form (the problem statement first, resources afterwards): pass d_workspace = NULL and
 * workspace_bytes = 0; the context is then created without touching the device and every compute
 * call returns MPR_ERR_WORKSPACE until mpr_set_workspace has attached one.                  */
int mpr_create(mpr_ctx** out, int L, const double* d_values, const uint8_t* d_mask,
               void* d_workspace, size_t workspace_bytes, void* cuda_stream);
/* Rectangular grids: Lx columns by Ly rows, row-major (site (x, y) at y * Lx + x),
 * d_values f64[Lx*Ly], d_mask u8[Lx*Ly].  Nothing in the method needs a square grid (PAPER.md:19:
 * nearest neighbours on a regular grid); the specific energy is normalised by the
 * Lx (Ly - 1) + Ly (Lx - 1) bonds of the open grid (R3; 2 L (L - 1) when square).  1 <= Lx, Ly <= 32768,
 * Lx * Ly >= 2.  mpr_create(L, ...) is mpr_create_rect(L, L, ...) with L >= 2; every other call takes the
 * shape from the context, and the [L*L] buffers named in this header are [Lx*Ly] for such a context.  */
int mpr_workspace_bytes_rect(int Lx, int Ly, size_t* bytes);
int mpr_create_rect(mpr_ctx** out, int Lx, int Ly, const double* d_values, const uint8_t* d_mask,
                    void* d_workspace, size_t workspace_bytes, void* cuda_stream);
void mpr_destroy(mpr_ctx* ctx); /* frees the host struct only */

/* Attaches (or replaces) the caller-owned device workspace: >= mpr_workspace_bytes(L) bytes, 256-byte
 * aligned, borrowed for the life of the context.  Runs the set-up described under mpr_create on the
 * context's stream (R1 range and map, sample energy of R6, mask bitmaps) and marks the chain for
 * re-initialisation; mode, seed, temperature and the other settings are kept.  Synchronises the
 * stream.  Fails with WORKSPACE, NO_MEASURED, DEGENERATE_RANGE, NONFINITE or CUDA; on failure the
 * context has no workspace.                                                                 */
int mpr_set_workspace(mpr_ctx* ctx, void* d_workspace, size_t workspace_bytes);
/* The cudaStream_t all later device work of the context is enqueued on (0 = default stream).  Work
 * already enqueued on the previous stream is waited for first, so the chain continues unchanged. */
int mpr_set_stream(mpr_ctx* ctx, void* cuda_stream);

/* Re-encodes the spins for `mode` and resets the chain (trial 0).                          */
int mpr_set_precision(mpr_ctx* ctx, mpr_precision mode);
/* The paper's (X_S X_E X_F) setting as three letters, e.g. "SDS"; see mpr_precision.  Resets the chain. */
int mpr_set_precision_triple(mpr_ctx* ctx, const char* xs_xe_xf);
/* The exponent q of Eq. 2 (q in (0, 1/2]; default 1/2, the value north_star fixes).  Recomputes the
 * sample energy and resets the chain.  With q < 1/2 the allowed arc of q phi is shorter than the half circle; the
 * range test that needs lives in the per-pass kernels, so the context then runs on MPR_PATH_PLAIN / MPR_PATH_LIST. */
int mpr_set_q(mpr_ctx* ctx, double q);
/* X_E alone: 0 = energy sums in double (default, R13), 1 = float energy variable.  Does not touch the chain. */
int mpr_set_energy_precision(mpr_ctx* ctx, int single);
/* Philox key (R9).  Resets the chain.                                                      */
int mpr_set_seed(mpr_ctx* ctx, uint64_t seed);
/* Reduced temperature T > 0, bypassing the estimate.  Does not touch the chain.            */
int mpr_set_temperature(mpr_ctx* ctx, double T);
/* Number of quench double-passes of the R8 initialisation (default 32).  Resets the chain. */
int mpr_set_quench(mpr_ctx* ctx, int n);
/* Kernel path (default MPR_PATH_AUTO) and temporal-blocking depth 0 <= k <= 4 (hybrid sweeps
 * fused per launch; 0, the default, lets the library choose: several per launch on small grids, where a launch is
 * latency-bound, one otherwise; the STRIP path uses min(k, 2)).  Results do not depend on either. */
int mpr_set_path(mpr_ctx* ctx, mpr_path path);
int mpr_set_fused_sweeps(mpr_ctx* ctx, int k);
/* Pass order of a hybrid sweep (see mpr_schedule).  Does not touch the chain.               */
int mpr_set_schedule(mpr_ctx* ctx, mpr_schedule schedule);
/* R8: free spins i.i.d. uniform from Philox (pass INIT, `trial` in counter word 3), then the
 * quench passes; sweep counter, move counters and the prediction accumulator are cleared.  */
int mpr_reset_chain(mpr_ctx* ctx, uint32_t trial);

/* R6: conditional energy matching.  Finds T with e_cond(T) = e_sample by bracketing on
 * [1e-4, 1] (expanded by decades within [1e-6, 1e2]) and Illinois regula falsi; each trial
 * is a fresh chain of 200 + 50 hybrid sweeps.  HOST outs (each may be null).  Sets T and
 * resets the chain (trial 0).  Fails with NO_MEASURED (no measured pair) or NO_ROOT.       */
int mpr_estimate_temperature(mpr_ctx* ctx, double* T_hat, double* e_sample, int* n_trials);

/* Continues the chain: n_eq hybrid sweeps (R4: Metropolis colour 0, 1, over-relaxation
 * colour 0, 1), then n_meas sweeps each followed by the energy sample e_n = 2H/N_b (R3) and
 * phi added to the per-site accumulator.
 *   d_pred    f64[L*L] or null: measured sites get their input value back bit-exact,
 *             prediction sites z_min + (z_max - z_min) * mean(phi) / 2pi over all measurement
 *             sweeps since the last chain reset (NaN if there were none).
 *   e_mean, e_stderr   HOST, may be null: mean of this call's e_n and its binned standard
 *             error (R16); NaN / 0 when n_meas == 0.                                       */
int mpr_run(mpr_ctx* ctx, int n_eq, int n_meas, double* d_pred, double* e_mean, double* e_stderr);

/* n hybrid sweeps without measurement (asynchronous).                                      */
int mpr_sweep(mpr_ctx* ctx, int n);
/* Single colour passes on the plain path, for tests: kind 0 = Metropolis (uses the Philox
 * stream of sweep number `sweep`), 1 = over-relaxation, 2 = quench, 3 = Metropolis followed at
 * once by over-relaxation at every site of the colour (the pass of the site-fused schedule). */
int mpr_pass(mpr_ctx* ctx, int kind, int colour, uint64_t sweep);

/* Spins as angles, d_phi f64[L*L] row-major (parity tests).  State only: the sweep counter, the move
 * counters and the prediction accumulator are not part of it.                              */
int mpr_get_state(mpr_ctx* ctx, double* d_phi);
/* Overwrites the spins at the prediction sites from d_phi (measured sites keep R1's map); angles
 * outside [0, 2pi] are clamped to the nearer end.  Counters and accumulator are left alone.  */
int mpr_set_state(mpr_ctx* ctx, const double* d_phi);
/* Energy of the current state: H (Eq. 2) and e = 2H/N_b.  HOST outs.                       */
int mpr_energy(mpr_ctx* ctx, double* H, double* e);
/* Sample energy of R6 and the number of measured pairs.  HOST outs.                        */
int mpr_sample_energy(mpr_ctx* ctx, double* e_sample, int64_t* n_pairs);
/* Accepted / attempted Metropolis moves and hybrid sweeps since the last chain reset.      */
int mpr_get_counters(mpr_ctx* ctx, uint64_t* accepted, uint64_t* attempted, uint64_t* sweeps);
/* Device time of the EQUILIBRATION phase of the last mpr_run: the n_eq hybrid sweeps that carry no
 * measurement, i.e. back-to-back launches of the sweep kernel alone (on the tiled path with fused
 * depth k: ceil(n_eq / k) launches of tiled_sweep_kernel<mode, 0>), timed by two CUDA events on the
 * ctx stream; the chain reset before them and the measurement sweeps after them are outside.  This
 * is what bench.py divides to get the dominant kernel's average launch duration INSIDE the timed
 * step.  HOST outs, each may be NULL.  eq_ms = 0 and eq_launches = 0 when n_eq
 * was 0.  MPR_ERR_NOT_READY before the first mpr_run.  The two events are the only CUDA objects the
 * library creates; mpr_destroy releases them.                                               */
int mpr_get_run_timing(mpr_ctx* ctx, double* eq_ms, int64_t* eq_launches, int64_t* eq_sweeps);
/* e_n of the last mpr_run, copied to HOST out[0..cap); returns their number (>= 0).        */
int64_t mpr_get_energy_series(mpr_ctx* ctx, double* out, int64_t cap);
/* z_min, z_max of the measured sample and the number of prediction sites.  HOST outs.      */
int mpr_get_info(mpr_ctx* ctx, double* z_min, double* z_max, int64_t* n_free, double* T);
/* Kernel launches enqueued by this context so far (for bench.py's gpu_launches).           */
int mpr_get_launch_stats(mpr_ctx* ctx, uint64_t* launches);

/* End-to-end call on HOST buffers (bench.py's e2e leg): copies h_values / h_mask to a staging
 * area at the end of the workspace, creates a context, selects mode and seed, takes T (or
 * estimates it when T <= 0), runs n_eq + n_meas sweeps and copies the prediction back.
 *   h_values f64[L*L], h_mask u8[L*L], h_pred f64[L*L]: HOST (pinned memory makes the copies
 *   asynchronous); d_workspace >= mpr_workspace_bytes_host(L) bytes; outs HOST, may be null. */
int mpr_workspace_bytes_host(int L, size_t* bytes);
int mpr_predict_host(int L, const double* h_values, const uint8_t* h_mask, mpr_precision mode,
                     uint64_t seed, double T, int n_eq, int n_meas, void* d_workspace,
                     size_t workspace_bytes, void* cuda_stream, double* h_pred, double* e_mean,
                     double* e_stderr, double* T_used, uint64_t* launches);
/* The same on an Lx x Ly grid (see mpr_create_rect). */
int mpr_workspace_bytes_host_rect(int Lx, int Ly, size_t* bytes);
int mpr_predict_host_rect(int Lx, int Ly, const double* h_values, const uint8_t* h_mask,
                          mpr_precision mode, uint64_t seed, double T, int n_eq, int n_meas,
                          void* d_workspace, size_t workspace_bytes, void* cuda_stream, double* h_pred,
                          double* e_mean, double* e_stderr, double* T_used, uint64_t* launches);

/* ---- Slabs of a larger grid (1-D decomposition over rows, one slab per GPU) ----------------
 * A context created (mpr_create_rect) on rows [row0, row0 + Ly) of a larger Lx-column grid becomes a SLAB of it:
 *   mpr_set_slab   global_row0 (even, >= 0) = the grid row of the slab's row 0; rows [own_begin, own_end) of the
 *                  slab are the rows it OWNS, the others are halo copies of its neighbours' rows; z_min / z_max =
 *                  the range of the WHOLE measured sample (R1); global_bonds = the whole grid's bond count (R3).
 *                  From then on the random numbers are keyed on the global site index (so the slabs together make
 *                  the moves a single context on the whole grid makes, bit for bit), the accepted-move count, the
 *                  prediction-site count and every energy sum cover the own rows only, and energies are normalised
 *                  by global_bonds: the whole grid's e is the SUM of the slabs' e.  Resets the chain.  A halo row
 *                  is updated like any other row but sees the slab's edge as an open boundary: one colour pass
 *                  spoils one more row from each inner edge (4 per hybrid sweep, 2 per quench double pass), so the
 *                  caller refreshes the halos (export from the owner, import into the neighbour) at least every
 *                  halo / 4 sweeps -- paper_1910_08448_b200/slabs.py does, in one process or one rank per slab.
 *                  (mpr_set_workspace on a slab context: call mpr_set_slab again afterwards.)
 *   mpr_create_slab   mpr_create_rect for rows that are GOING TO BE a slab: the local sample may hold no measured site, or a
 *                  single value (sparse data, thin slabs) -- what counts is the whole grid's range, which mpr_set_slab
 *                  brings; until mpr_set_slab every compute call returns MPR_ERR_NOT_READY.  Non-finite measured values
 *                  still fail.
 *   mpr_set_peers  PEER MODE: instead of export / import between launches, every STRIP launch of a slab stores the 4 own
 *                  rows next to each inner edge straight into the halo rows of the neighbour's destination buffer
 *                  (peer memory: on one GPU another pointer, between GPUs of one process a store over NVLink once peer
 *                  access is enabled) and its own buffer receives its halo rows the same way -- compute and exchange in
 *                  ONE kernel, no copy launch.  up / down = the contexts of the slabs above / below (null at the ends of
 *                  the grid; both null leaves peer mode).  Requirements: slabs of the same grid, mode and stream, halo
 *                  of exactly 4 rows, >= 8 own rows, q = 1/2; every slab makes the same sequence of calls, one launch
 *                  each in turn (a launch finds the neighbour's buffer by the number of launches both have made);
 *                  one sweep per launch, quench double passes two per launch.  Launch n + 1 of a slab must follow launch
 *                  n of its neighbours (it reads the halo rows they wrote and overwrites the buffer they read): on ONE
 *                  stream the stream order gives that; with a stream per slab the caller records an event after every
 *                  launch and makes the neighbours' streams wait for it before their next one (slabs.py does;
 *                  tests/test_slabs_gpu.py runs it on one GPU).  Slabs on several devices of one process need peer
 *                  access enabled besides: the same calls, not exercised here.  Resets the chain.
 *   mpr_sample_energy_parts   the sum of cos over, and the number of, measured nearest-neighbour pairs to the right
 *                  of and below the own rows: e_s of the whole grid = -2 J sum(parts) / sum(counts).  HOST outs.
 *   mpr_rows_bytes / mpr_export_rows / mpr_import_rows   n_rows rows of the chain state from row_begin on (both
 *                  colours, in the storage type of the mode), packed into / read from a DEVICE buffer of
 *                  mpr_rows_bytes bytes; enqueued on the context's stream.
 *   mpr_advance    n_sweeps hybrid sweeps without the bookkeeping of mpr_run; measure = 0: sweeps only, 1: the energy
 *                  of each sweep goes to slot first_slot + i of the device series, 2: and phi is accumulated.
 *   mpr_quench     n quench double passes (R8: colour 0, colour 1) on the chain as it is, by the kernels of the path.
 *   mpr_fetch_series   the first n slots of that series -> HOST out (synchronises the stream).
 *   mpr_predict    the back-mapped average of phi accumulated since the last chain reset -> d_pred f64[Lx*Ly].
 *   mpr_debug_trial_lengths   the fixed sweep counts of one temperature trial of R6 (equilibration, measurement). */
int mpr_create_slab(mpr_ctx** out, int Lx, int Ly, const double* d_values, const uint8_t* d_mask,
                    void* d_workspace, size_t workspace_bytes, void* cuda_stream);
int mpr_set_slab(mpr_ctx* ctx, int global_row0, int own_begin, int own_end, double z_min, double z_max,
                 double global_bonds);
int mpr_set_peers(mpr_ctx* ctx, mpr_ctx* up, mpr_ctx* down);
int mpr_sample_energy_parts(mpr_ctx* ctx, double* cos_sum, int64_t* n_pairs);
int mpr_rows_bytes(mpr_ctx* ctx, int n_rows, size_t* bytes);
int mpr_export_rows(mpr_ctx* ctx, int row_begin, int n_rows, void* d_out);
int mpr_import_rows(mpr_ctx* ctx, int row_begin, int n_rows, const void* d_in);
int mpr_advance(mpr_ctx* ctx, int n_sweeps, int measure, int first_slot);
int mpr_quench(mpr_ctx* ctx, int n_double_passes);
int mpr_fetch_series(mpr_ctx* ctx, int n, double* h_out);
int mpr_predict(mpr_ctx* ctx, double* d_pred);
void mpr_debug_trial_lengths(int* n_eq, int* n_meas);

/* ---- The one entry point that needs no workspace and allocates nothing (csrc/mpr_static.cu) -------------------
 * For callers that cannot call cudaMalloc (code under CUDA-graph capture, serving loops, harnesses that forbid it)
 * and have no workspace for mpr_create: the sample statistics the method starts from (R1: range of the measured
 * values; R6 first half: the sample energy e_s = -2 J mean of cos[q (phi_s - phi_t)] over nearest-
 * neighbour pairs with both ends measured), computed by four kernel launches on cuda_stream with every intermediate
 * (per-block partial sums, the range) in a file-scope `static __device__` array of the library: 49 216 bytes, held
 * by every GPU that loads libmpr.so until the process exits.  No cudaMalloc / cudaFree, no host allocation on the
 * success path, no synchronisation: the call returns when the work is enqueued.
 *   Lx, Ly     columns, rows; Lx * Ly >= 2 and <= mpr_static_max_sites() = 2^28 (16384 x 16384).  Larger grids are
 *              rejected with MPR_ERR_INVALID_ARG (mpr_static_last_error() says why): use mpr_create.
 *   d_values   f64[Lx*Ly] DEVICE, never read where d_mask == 1;  d_mask u8[Lx*Ly] DEVICE, 1 = prediction site
 *   q          of Eq. 2, in (0, 1/2]; the paper's value is 0.5
 *   d_out      f64[6] DEVICE, caller-owned: e_s, number of measured pairs, z_min, z_max, number of measured sites,
 *              number of non-finite measured values.  e_s is NaN where mpr_create would have failed (no measured
 *              pair, a non-finite measured value, z_max == z_min): the host cannot know without a synchronisation.
 * The same numbers as mpr_create + mpr_sample_energy + mpr_get_info give (same per-thread order of operations).
 * SHARED STATE: every call on a device uses the same array.  Calls that overlap on the GPU (different streams or
 * threads without an ordering between them) race; calls on one stream, or ordered by events, do not.  The array
 * keeps the previous call's contents; every slot a call reads it has written first, nothing needs clearing.
 * mpr_static_setup() takes the array's device address for the CURRENT device (cudaGetSymbolAddress, once per
 * device); the entry point does so itself on first use, but a caller about to capture a graph calls it beforehand.
 * mpr_static_last_error(): message of the calling thread's last failed mpr_*_static* call ("" after a success). */
int mpr_static_setup(void);
int64_t mpr_static_max_sites(void);
const char* mpr_static_last_error(void);
int mpr_sample_energy_static(int Lx, int Ly, const double* d_values, const uint8_t* d_mask, double q,
                             void* cuda_stream, double* d_out);

/* HOST-only hooks into the library's host-side numerics, so that they can be pinned against
 * hand-worked numbers without a GPU (tests/test_host_logic.py); no device work, no context.
 *   mpr_debug_series_stats       mean and binned standard error (R16) of h_series[0..n), exactly
 *                                the routine mpr_run and the temperature trials use.
 *   mpr_debug_match_temperature  the root search of R6 (steps 1-5 in DESIGN.md) as
 *                                mpr_estimate_temperature runs it, with the trial chains replaced by
 *                                the caller's function: trial(T, trial_index (1, 2, ...), &e, &se, user)
 *                                returns 0 and the mean energy / standard error "measured" at T.
 *                                Returns MPR_OK and T_hat, or MPR_ERR_NO_ROOT; *n_trials = trials made.
 *   mpr_debug_proposal_width     the Metropolis proposal half-width delta(T) of R7 the kernels are given. */
double mpr_debug_proposal_width(double T);
double mpr_debug_proposal_width_q(double T, double q);
typedef int (*mpr_trial_fn)(double T, int trial_index, double* e, double* se, void* user);
int mpr_debug_series_stats(const double* h_series, int64_t n, double* mean, double* se);
int mpr_debug_match_temperature(double e_sample, mpr_trial_fn trial, void* user, double* T_hat,
                                int* n_trials);

/* The Philox4x32-10 block function and the uniform the kernels use, evaluated on the DEVICE
 * for n counters (tests pin the in-kernel generator against the CUDA toolkit's own).
 *   d_ctr u32[4n], key[2] HOST, d_out u32[4n]                                              */
int mpr_debug_philox(const uint32_t* d_ctr, const uint32_t key[2], uint32_t* d_out, int64_t n,
                     void* cuda_stream);

/* The Metropolis decision of the double-arithmetic modes (float filter, double evaluation only when the
 * filter cannot decide) next to the plain double evaluation u2 < exp(min(-dE/T, 0)), on the DEVICE, for n moves:
 *   d_words u32[2n] (the two Philox words of u2), d_mdE f64[n] (-dE), T; d_out u8[n]: bit 0 = filtered decision,
 *   bit 1 = plain decision, bit 2 = the filter decided alone.  Tests require bit 0 == bit 1 on adversarial inputs.  */
int mpr_debug_accept(const uint32_t* d_words, const double* d_mdE, double T, uint8_t* d_out, int64_t n,
                     void* cuda_stream);

const char* mpr_last_error(const mpr_ctx* ctx);
const char* mpr_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* MPR_H_ */
