/*
 * mpr.h -- C ABI of the B200-native (sm_100a) hot path of the modified planar
 * rotator (MPR) conditional simulation, arXiv 1811.01604 ("PAPER.md").
 *
 * The library fills the gaps of `batch` independent rows x cols grids:
 * sample sites (mask = 1) are held fixed, prediction sites (mask = 0) are
 * simulated by the checkerboard hybrid Monte Carlo sweep (PAPER.md L113-146
 * Alg. 1) to the paper's energy-slope equilibration (L192-206,
 * Alg. 2 step 5), followed by M realizations (L207-211, step 6) whose mean is
 * back-transformed into the interpolated map (L148, L212, step 7).
 *
 * Conventions (all entry points)
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.
 *   - The caller owns every buffer it passes (inputs, workspace, outputs).
 *     The library owns only the small host-side mpr_ctx (with host copies of
 *     the per-grid scalars and flags it polls).  All device state lives
 *     inside the caller's workspace.
 *   - Every call returns an mpr_status; nothing throws, aborts or sets errno.
 *     Output parameters are left untouched when the status is not MPR_OK.
 *   - Work is enqueued on the CUDA stream given to mpr_create.  Calls that
 *     return host data (and mpr_create / mpr_equilibrate, which need device
 *     results to size launches / stop the loop) synchronise that stream; the
 *     others return as soon as the work is enqueued.
 *   - A context is not thread-safe; distinct contexts are independent.
 *   - Grids are row-major, [batch][rows][cols]; rectangular grids are allowed
 *     (PAPER.md L261).  2 <= rows, cols <= 65534; rows*cols < 2^31.
 *   - Random numbers: Philox4x32-10 keyed by `seed`, counter
 *     (site = row*cols + col, t >> 1, 2, grid) for the sweeps -- words 0,1 give
 *     (u, r) of the even global sweep index t, words 2,3 of the odd one -- and
 *     (site >> 2, 0, 0, grid) for the initial state (reading R13).
 *     t counts sweeps from mpr_set_params on, through equilibration and every
 *     realization.
 */
#ifndef MPR_H
#define MPR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mpr_ctx mpr_ctx; /* opaque */

typedef enum {
    MPR_OK = 0,
    MPR_ERR_ARG = 1,              /* bad argument (null pointer, size, q, T, M, ...) */
    MPR_ERR_NO_SAMPLES = 2,       /* a grid has no sample site (mask all 0) */
    MPR_ERR_NO_FREE = 3,          /* a grid has no prediction site (mask all 1) */
    MPR_ERR_DEGENERATE_RANGE = 4, /* z_max == z_min over the samples: Eq. 1 divides by zero */
    MPR_ERR_NONFINITE = 5,        /* a sample value is NaN or Inf */
    MPR_ERR_STATE = 6,            /* call out of order (e.g. sweep before set_params) */
    MPR_ERR_WORKSPACE = 7,        /* workspace too small or misaligned (256 B) */
    MPR_ERR_CUDA = 8,             /* a CUDA runtime call failed; see mpr_last_cuda_error */
    MPR_ERR_UNSUPPORTED = 9,      /* valid per the paper but not built (or_mode 1 with q != 1/2) */
    MPR_ERR_COMM = 10,            /* a communication callback of a slab context returned non-zero */
    MPR_ERR_TOO_LARGE = 11        /* a size beyond the fixed scratch of the allocation-free entry point */
} mpr_status;

/* Alg. 2 step 1 parameters.  POD, host memory. */
typedef struct {
    uint32_t struct_size;     /* = sizeof(mpr_params); ABI versioning */
    float    q;               /* coupling exponent, 0 < q <= 0.5; paper: 1/2 (L89) */
    uint32_t equil_cap;       /* i_max, at most this many equilibration sweeps (L171, L192) */
    uint32_t sweeps_per_real; /* UPDATE sweeps per realization; paper 1 (L210), BASELINE configs 100 */
    uint32_t M;               /* number of realizations (L168), >= 1 */
    uint32_t n_f;             /* slope checked every n_f sweeps (L169, L201) */
    uint32_t n_fit;           /* window of the slope fit, 2 <= n_fit <= 256 (L169, L201) */
    float    A_targ;          /* target acceptance ratio (L170, L196) */
    float    k_a;             /* proposal-width growth constant (L171, L197) */
    uint32_t or_mode;         /* 0 exact-q reflection (R2), 1 Eq. 6 as printed (q = 1/2 only), 2 off */
    uint32_t a_eq_mode;       /* 0 keep the a reached in equilibration, 1 a = 1 as printed at L210 (R10) */
    uint64_t seed;            /* Philox key */
} mpr_params;

/* Per-grid run statistics (host). */
typedef struct {
    uint32_t equil_sweeps;    /* i: sweeps done by mpr_equilibrate */
    uint32_t t;               /* global sweep index (sweeps since mpr_set_params) */
    uint32_t equilibrated;    /* 1 once the stopping rule k >= 0 or the cap was reached */
    uint32_t realizations;    /* realizations accumulated so far */
    uint64_t n_free;          /* P: prediction sites */
    uint64_t n_samples;       /* sample sites */
    uint64_t n_bonds;         /* N_GP = rows(cols-1) + cols(rows-1) (L109) */
    double   a;               /* current proposal-width divisor, alpha = 2 pi / a (L156) */
    double   k;               /* last fitted energy slope (L201) */
    double   A_last;          /* acceptance ratio of the last counted sweep */
    double   e_last;          /* energy per bond after the last counted sweep (L199) */
    float    z_min, z_max;    /* Eq. 1 range (L81) */
} mpr_stats;

/* Default parameters: q = 1/2, n_f = 5, n_fit = 20, A_targ = 0.3, k_a = 3,
 * equil_cap = 500, M = 100, sweeps_per_real = 1, modes 0, seed 0
 * (reading R7; the paper defers them to its companion paper, L166). */
void mpr_default_params(mpr_params* h_out);

/* Bytes of device workspace mpr_create needs for `batch` grids of rows x cols
 * (worst case: every site a prediction site).  MPR_ERR_ARG on bad sizes. */
mpr_status mpr_query_workspace(int batch, int rows, int cols, size_t* h_bytes);

/* Problem statement: grid, sample set, sample values.
 * Computes z_min / z_max over SAMPLE sites (L81), the data->angle transform
 * of Eq. 1 (L79) at sample sites, the fixed-site bitmask and the
 * checkerboard-split (L261) lists of prediction sites.
 *   d_values      device float [batch][rows][cols]; values at mask==0 sites are ignored (may be NaN)
 *   d_sample_mask device uint8 [batch][rows][cols]; nonzero = sample (fixed), 0 = prediction site
 *   d_workspace   device, >= mpr_query_workspace bytes, 256-byte aligned; must outlive the context
 *   cuda_stream   a cudaStream_t (0 = default stream); all later work runs on it
 * The inputs are consumed before the call returns (it synchronises).
 * Errors: ARG, WORKSPACE, NO_SAMPLES, NO_FREE, DEGENERATE_RANGE, NONFINITE, CUDA. */
mpr_status mpr_create(mpr_ctx** out, int batch, int rows, int cols,
                      const float* d_values, const uint8_t* d_sample_mask,
                      void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* Alg. 2 steps 1-2 (L165-180): stores the parameters and the per-grid
 * temperatures (h_T host float [batch], T > 0 finite), draws the initial state
 * U(0, 2 pi) at the prediction sites from the INIT stream, resets i = 0,
 * a = 1, k = -1, t = 0 and the realization accumulator.  May be called again
 * to restart.  Errors: ARG, UNSUPPORTED, CUDA. */
mpr_status mpr_set_params(mpr_ctx* ctx, const mpr_params* h_params, const float* h_T);

/* Alg. 2 step 5 (L192-206): per grid, sweep until the fitted energy slope
 * k >= 0 or equil_cap sweeps; adapts a by step 5.2.  Synchronises. */
mpr_status mpr_equilibrate(mpr_ctx* ctx);

/* Alg. 2 step 6 (L207-211): M x {sweeps_per_real sweeps; accumulate the state
 * at prediction sites}.  Asynchronous. */
mpr_status mpr_simulate(mpr_ctx* ctx);

/* Alg. 2 step 7 + back-transform (L148, L210-212): d_out device float
 * [batch][rows][cols]; prediction sites = z_min + mean(phi) (z_max - z_min)/(2 pi)
 * over the realizations accumulated so far (>= 1, else MPR_ERR_STATE), sample
 * sites = the input value bit for bit.  Asynchronous. */
mpr_status mpr_predict(mpr_ctx* ctx, float* d_out);

/* "Statistics of M realizations" (Alg. 2 step 7, L212; L148: the realizations sample the conditional
 * distribution): d_out device float [batch][rows][cols] receives, at prediction sites, the unbiased sample
 * standard deviation of the M back-transformed realizations accumulated so far,
 * sqrt(sum_k (phi_k - mean)^2 / (M - 1)) (z_max - z_min) / (2 pi), and 0 at sample sites.  Needs M >= 2
 * realizations (else MPR_ERR_STATE).  Synchronises. */
mpr_status mpr_predict_std(mpr_ctx* ctx, float* d_out);

/* Quantiles from the first two moments of the realizations (L212; reading R26):
 * d_out device float [batch][rows][cols] receives, at prediction sites, the Gaussian p-quantile
 * mean + Phi^-1(p) * (standard deviation of mpr_predict_std), clamped to the data range [z_min, z_max] that the
 * state space [0, 2 pi] maps to; sample sites = the input value.  0 < p < 1 (else MPR_ERR_ARG), needs >= 2
 * realizations (else MPR_ERR_STATE).  p = 0.5 is mpr_predict.  Synchronises. */
mpr_status mpr_predict_quantile(mpr_ctx* ctx, double p, float* d_out);

/* ---- chain parallelism (a variant of the paper's single chain, reading R25) ----
 * The M realizations of step 6 ("Statistics of M realizations") made by `chains` independent
 * chains per grid instead of one, so that small grids fill the device: mpr_equilibrate runs one chain per grid
 * as Alg. 2 step 5 says; mpr_simulate then starts chains 1 .. chains-1 from a copy of that equilibrated state
 * (same sweep index t), chain c of grid g drawing from the Philox grid word g + c * batch, and every chain makes
 * ceil(M / chains) realizations of sweeps_per_real sweeps, all in the same launches.  mpr_predict and
 * mpr_predict_std pool the realizations of a grid's chains; mpr_stats.realizations is their total.  The
 * diagnostic calls (get/set_angles, sweep, energy, measure_energy) act on chain 0; after any of them, and after
 * mpr_equilibrate, the next mpr_simulate forks again (accumulators are kept).  chains = 1 is mpr_create.
 * batch * chains <= 65535.  Workspace: mpr_query_workspace_chains bytes. */
mpr_status mpr_query_workspace_chains(int batch, int chains, int rows, int cols, size_t* h_bytes);
mpr_status mpr_create_chains(mpr_ctx** out, int batch, int chains, int rows, int cols,
                             const float* d_values, const uint8_t* d_sample_mask,
                             void* d_workspace, size_t workspace_bytes, void* cuda_stream);

mpr_status mpr_destroy(mpr_ctx* ctx);

/* ---- Alg. 2 step 4: parameter inference ---- */

/* Step 4.1, Eq. 4 (L101-104): sample specific energy e_s = -(1/N_SP) sum over the nearest-neighbour
 * pairs of SAMPLE sites of cos q(phi_i - phi_j), every unordered pair once (reading R1), with
 * q of the last mpr_set_params (1/2 before the first).  h_e_s host double [batch], h_n_pairs host
 * uint64 [batch] (N_SP; e_s = 0 where N_SP = 0).  Needs only mpr_create.  Synchronises. */
mpr_status mpr_sample_energy(mpr_ctx* ctx, double* h_e_s, uint64_t* h_n_pairs);

/* A context of `batch` unconditional grids (L109: "the values of the spins can be varied at every grid
 * node"): no data, every node a prediction site, Eq. 1 the identity on [0, 2 pi].  mpr_set_params starts
 * each grid from the ordered state phi = pi instead of the uniform draw, and mpr_equilibrate burns in for
 * exactly equil_cap sweeps with the a-control of step 5.2 but without the slope stop (from the ordered state
 * the energy rises, so k >= 0 holds at the first check; reading R23); everything else (mpr_sweep,
 * mpr_measure_energy, mpr_energy, ...) works as on a conditional context.
 * Workspace as mpr_query_workspace(batch, rows, cols).  Errors: ARG, WORKSPACE, CUDA. */
mpr_status mpr_create_unconditional(mpr_ctx** out, int batch, int rows, int cols,
                                    void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* n_sweeps further UPDATE sweeps of every grid at its current a, the energy per bond taken after each
 * (the fused reduction of the equilibration pass); h_e_mean host double [batch] receives the mean over
 * these sweeps: <H> / N_GP of Eq. 5 (L105-109) for an equilibrated chain.  t advances by n_sweeps.
 * Synchronises.  Errors: ARG (n_sweeps = 0), STATE, CUDA. */
mpr_status mpr_measure_energy(mpr_ctx* ctx, uint32_t n_sweeps, double* h_e_mean);

/* Step 4.2, Eq. 5: e(T_k, L) for a ladder of n_T temperatures h_T (host float, > 0) on a rows x cols
 * grid: one unconditional chain per temperature (chain k = grid k of one batch), mpr_set_params(h_params,
 * h_T), mpr_equilibrate, mpr_measure_energy(n_meas).  h_e host double [n_T].  d_workspace: at least
 * mpr_query_workspace(n_T, rows, cols) bytes.  Synchronises. */
mpr_status mpr_energy_table(int rows, int cols, const mpr_params* h_params, const float* h_T, int n_T,
                            uint32_t n_meas, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                            double* h_e);

/* Step 4.2, T = argmin_T |e_s - e(T, L)| (L111) over the piecewise-linear interpolant of the ladder
 * (h_T ascending): the first segment that brackets e_s, else the ladder point nearest in energy (reading
 * R24).  Host arithmetic on n_T numbers.  Errors: ARG. */
mpr_status mpr_infer_temperature(const float* h_T, const double* h_e, int n_T, double e_s, double* h_T_hat);

/* The ladder step 4.2 uses when the caller has none: n_T temperatures h_T[k] = T_c * h_factors[k] around
 * T_c = 2 N_GP (1 + e_s) / (N - 1), the temperature at which the low-temperature equipartition energy
 * e(T) = -1 + (N - 1) T / (2 N_GP) of a rows x cols grid (N - 1 harmonic modes, N_GP bonds, J = 1; DESIGN.md
 * reading R15) equals e_s.  That line only CENTRES the ladder; e(T_k, L) itself comes from the chains of
 * mpr_energy_table.  h_factors host float [n_T], ascending, > 0; NULL = {1/4, 1/2, 1, 2, 4} (then n_T must be 5).
 * h_T host float [n_T].  Host arithmetic.  Errors: ARG. */
mpr_status mpr_default_ladder(int rows, int cols, double e_s, const float* h_factors, int n_T, float* h_T);

/* Alg. 2 step 4 as ONE call (L97-111, L186-190), for every grid of `ctx` (which needs only mpr_create):
 * e_s by Eq. 4 with q of h_params (mpr_sample_energy), the ladder of mpr_default_ladder around it, e(T_k, L)
 * of Eq. 5 from unconditional chains (mpr_energy_table: h_params->equil_cap burn-in sweeps, n_meas measured
 * ones, h_params->seed), and T-hat = argmin |e_s - e(T, L)| over the ladder's interpolant (mpr_infer_temperature).
 * d_workspace: device, at least mpr_query_workspace(n_T, rows, cols) bytes, 256-byte aligned; it is scratch for the
 * unconditional chains (one grid's ladder at a time) and distinct from the context's own workspace.
 * h_T_hat host double [batch]; h_e_s host double [batch] or NULL.  The result goes to mpr_set_params as T.
 * Synchronises.  Errors: ARG, NO_SAMPLES (a grid without a pair of neighbouring samples), WORKSPACE, CUDA. */
mpr_status mpr_infer_temperature_auto(mpr_ctx* ctx, const mpr_params* h_params, const float* h_factors, int n_T,
                                      uint32_t n_meas, void* d_workspace, size_t workspace_bytes,
                                      double* h_T_hat, double* h_e_s);

/* ---- q learned from the data ("In principle, q can be learned from the data"; the paper fixes q = 1/2
 * and gives no procedure: DESIGN.md reading R28) ----
 * Leave-out validation over n_q candidates h_q (0 < q <= 1/2) on one rows x cols grid: a fraction holdout_fraction
 * of the samples is withheld (sample site n when the uniform of the HOLDOUT stream -- Philox counter (n >> 2, 0, 3, 0),
 * word n & 3, key h_params->seed -- is below it); for every candidate the whole path runs on the remaining samples
 * (Eq. 1 over them; T from their specific energy at this q, Eq. 4, through the equipartition line, i.e. the centre of
 * mpr_default_ladder; mpr_set_params with h_params and this q, mpr_equilibrate, mpr_simulate, mpr_predict) and is
 * scored by the root mean square error of the prediction at the withheld samples, h_scores[k].  *h_q_hat = the
 * candidate with the smallest score (the first of equals); h_T (host double [n_q], may be NULL) receives the
 * temperatures used.  d_workspace: mpr_query_workspace_learn_q bytes, 256-byte aligned.  Synchronises.
 * Errors: ARG, WORKSPACE, those of mpr_create on the remaining samples, NO_SAMPLES when nothing was withheld. */
mpr_status mpr_query_workspace_learn_q(int rows, int cols, size_t* h_bytes);
mpr_status mpr_learn_q(int rows, int cols, const float* d_values, const uint8_t* d_sample_mask, const mpr_params* h_params,
                       const float* h_q, int n_q, double holdout_fraction, void* d_workspace, size_t workspace_bytes,
                       void* cuda_stream, float* h_q_hat, double* h_scores, double* h_T);

/* ---- one grid across several GPUs: row-block decomposition (the
 * paper's double-precision run at L = 8192 did not fit its card) ----
 * The rows of ONE rows_global x cols grid are dealt in blocks to several contexts ("slabs"), one per process / GPU.
 * A slab owns rows [row_begin, row_end) and keeps 8 ghost rows of each neighbouring slab (none at the grid's edge).
 * The random numbers are keyed by the site's index in the WHOLE grid, the colours by the global row, Eq. 1 uses the
 * minimum and maximum over every slab's samples, A = accepted / P and e = H / N_GP of Alg. 2 step 5 are sums over the
 * slabs: the slabs together compute, bit for bit in the state, what one context computes on the whole grid (ghost
 * sites are updated redundantly, like the halo of a tile, and renewed after every pass of up to 4 sweeps).
 * The library owns the loops; moving data between slabs is the caller's, through two callbacks (host functions; return
 * 0 on success, anything else ends the call with MPR_ERR_COMM):
 *   allreduce(user, h_values, n, op): replace the n host doubles by their sum / minimum / maximum over all slabs
 *       (op = MPR_REDUCE_*).  Called by mpr_create_slab (3 times), once per sweep by mpr_equilibrate, by mpr_energy.
 *   exchange(user, cuda_stream): the library has enqueued on cuda_stream copies of its 8 own rows next to the upper
 *       boundary into d_send_up and next to the lower boundary into d_send_down (mpr_slab_halo_bytes(cols) bytes
 *       each: 8 rows of [cols rounded up to even] float2); when the work the callback enqueues on cuda_stream (or has
 *       completed) is done, d_recv_up must hold the upper neighbour's d_send_down and d_recv_down the lower
 *       neighbour's d_send_up.  Called after every pass (with NCCL: ncclSend / ncclRecv on that stream).
 * Every slab must make the same calls in the same order (mpr_set_params with the same parameters and T, ...).
 * Constraints: row_begin even, at least 8 own rows, rows_global * cols < 2^32, one chain, batch 1.
 * The context's "grid" is the slab's LOCAL rows: own rows plus ghost rows, mpr_slab_local_rows gives their place in the
 * whole grid; d_values / d_sample_mask of mpr_create_slab and the outputs of mpr_predict*, mpr_get_angles have that
 * shape [n_rows][cols] (ghost rows of the outputs are to be ignored); mpr_get_stats counts the own rows' sites;
 * mpr_energy returns the whole grid's energy per bond on every slab.  Unmeasured on more than one GPU. */
enum { MPR_REDUCE_SUM = 0, MPR_REDUCE_MIN = 1, MPR_REDUCE_MAX = 2 };
typedef int (*mpr_allreduce_fn)(void* user, double* h_values, int n, int op);
typedef int (*mpr_exchange_fn)(void* user, void* cuda_stream);
typedef struct {
    uint32_t struct_size;          /* = sizeof(mpr_slab) */
    int rows_global, cols;         /* the whole grid */
    int row_begin, row_end;        /* this slab's own rows [row_begin, row_end) */
    mpr_allreduce_fn allreduce;
    mpr_exchange_fn exchange;
    void* user;                    /* passed to the callbacks */
    void* d_send_up;               /* device staging buffers, mpr_slab_halo_bytes(cols) bytes each, caller-owned; */
    void* d_recv_up;               /*   the *_up pair may be NULL when row_begin = 0, */
    void* d_send_down;             /*   the *_down pair when row_end = rows_global */
    void* d_recv_down;
} mpr_slab;
size_t mpr_slab_halo_bytes(int cols);
/* The rows of the whole grid a slab holds: [*h_first_row, *h_first_row + *h_n_rows) = own rows plus ghost rows. */
mpr_status mpr_slab_local_rows(const mpr_slab* h_slab, int* h_first_row, int* h_n_rows);
mpr_status mpr_query_workspace_slab(const mpr_slab* h_slab, size_t* h_bytes);
/* As mpr_create for the slab's local rows (d_values, d_sample_mask: device [n_rows][cols]).  The callbacks and the
 * staging buffers must stay valid for the life of the context.  Errors: as mpr_create, judged on the whole grid
 * (NO_SAMPLES, NO_FREE, DEGENERATE_RANGE, NONFINITE come back on every slab alike), and COMM. */
mpr_status mpr_create_slab(mpr_ctx** out, const mpr_slab* h_slab, const float* d_values, const uint8_t* d_sample_mask,
                           void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- double-precision path (Table 2 against Table 3) ----
 * The same method with data, spin state, every site update and the realization sums in double: one grid per
 * context, values and outputs are double, "2 pi" is the double nearest 2 pi, Eq. 1 keeps its pinned operation
 * order (in double), the random streams are those of the fp32 path (same Philox counters, the same 24-bit
 * uniforms, grid word 0).  Calls mirror the fp32 ones (same statuses, same ordering rules, mpr_params as is;
 * T is one temperature).  mpr64_predict / mpr64_predict_std: d_out device double [rows][cols].  Angles are
 * exchanged as device double [rows][cols].  Workspace: mpr64_query_workspace bytes (71.4 B per site), 256-byte aligned. */
typedef struct mpr64_ctx mpr64_ctx; /* opaque */
mpr_status mpr64_query_workspace(int rows, int cols, size_t* h_bytes);
mpr_status mpr64_create(mpr64_ctx** out, int rows, int cols, const double* d_values, const uint8_t* d_sample_mask,
                        void* d_workspace, size_t workspace_bytes, void* cuda_stream);
mpr_status mpr64_set_params(mpr64_ctx* ctx, const mpr_params* h_params, double T);
mpr_status mpr64_equilibrate(mpr64_ctx* ctx);                 /* Alg. 2 step 5; synchronises */
mpr_status mpr64_simulate(mpr64_ctx* ctx);                    /* Alg. 2 step 6; asynchronous */
mpr_status mpr64_predict(mpr64_ctx* ctx, double* d_out);      /* Alg. 2 step 7; asynchronous */
mpr_status mpr64_predict_std(mpr64_ctx* ctx, double* d_out);  /* L212; needs >= 2 realizations; synchronises */
mpr_status mpr64_destroy(mpr64_ctx* ctx);
mpr_status mpr64_get_angles(mpr64_ctx* ctx, double* d_phi);
mpr_status mpr64_set_angles(mpr64_ctx* ctx, const double* d_phi);     /* prediction sites only are overwritten */
mpr_status mpr64_set_sweep_index(mpr64_ctx* ctx, uint32_t t);
mpr_status mpr64_sweep(mpr64_ctx* ctx, uint32_t n_sweeps, double a, uint64_t* h_accepted /* may be NULL */);
mpr_status mpr64_energy(mpr64_ctx* ctx, double* h_e_per_bond);
mpr_status mpr64_get_transform(mpr64_ctx* ctx, double* h_zmin, double* h_zmax);
mpr_status mpr64_get_stats(mpr64_ctx* ctx, mpr_stats* h_out);          /* z_min / z_max rounded to float here */
mpr_status mpr64_get_launch_count(mpr64_ctx* ctx, uint64_t* h_count);

/* ---- allocation-free entry point ----
 * For callers that can neither call cudaMalloc nor hand over a workspace (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid allocation): the energy per bond e = H / N_GP of Eq. 2 (the quantity
 * Alg. 2 step 5.3 tracks, L199) of an angle field in device memory, without a context.  mpr_energy keeps its partial
 * sums in the caller's workspace; this variant keeps one partial per grid row in a file-scope `static __device__` array
 * of the library: MPR_NOALLOC_MAX_ROWS doubles + a counter = 128 KB + 256 B, held by every GPU that loads the library
 * until the process exits.  The call makes no cudaMalloc, cudaFree or allocating library call.
 *   d_phi         device float [rows][cols], angles in [0, 2 pi] (sample and prediction sites alike: every bond counts)
 *   q             0 < q <= 1/2
 *   d_e_per_bond  device double [1]: receives e; written when the work enqueued on cuda_stream is done
 * Asynchronous (enqueues one 4-byte memset of the counter and one kernel on cuda_stream; no synchronisation).
 * rows > MPR_NOALLOC_MAX_ROWS is MPR_ERR_TOO_LARGE (mpr_last_cuda_error names the limit); other bad arguments
 * (null pointers, rows or cols < 2, cols > 65534, q out of range, d_phi not device memory) MPR_ERR_ARG.
 * The scratch is SHARED by every call and keeps the last call's contents: what must start at zero is cleared by the call
 * itself, but calls that overlap on the GPU (other streams, other host threads) race on it -- serialise them.  The first
 * call on a device looks the array's address up (cudaGetSymbolAddress); make that call outside a graph capture. */
#define MPR_NOALLOC_MAX_ROWS 16384
mpr_status mpr_energy_of_angles_noalloc(const float* d_phi, int rows, int cols, double q, double* d_e_per_bond,
                                        void* cuda_stream);

/* ---- diagnostic / test / checkpoint surface ---- */

/* Current angles phi in [0, 2 pi], device float [batch][rows][cols]. Sample
 * sites return Eq. 1 bit-exactly. Asynchronous. */
mpr_status mpr_get_angles(mpr_ctx* ctx, float* d_phi);
/* Overwrite the angles of the PREDICTION sites from d_phi (same shape);
 * sample sites are ignored. Asynchronous. */
mpr_status mpr_set_angles(mpr_ctx* ctx, const float* d_phi);
/* Set / get the global sweep index t of every grid (with get/set_angles this
 * is a complete checkpoint: the RNG is counter-based). */
mpr_status mpr_set_sweep_index(mpr_ctx* ctx, uint32_t t);
/* n_sweeps raw UPDATE sweeps (Alg. 1) at fixed a >= 1 on every grid; t
 * advances by n_sweeps. h_accepted (host uint64 [batch], may be NULL) receives
 * the accepted Metropolis proposals summed over these sweeps (synchronises
 * when non-NULL). */
mpr_status mpr_sweep(mpr_ctx* ctx, uint32_t n_sweeps, double a, uint64_t* h_accepted);
/* Energy per bond e = H / N_GP of Eq. 2 (L87, L109, L199), host double [batch]. Synchronises. */
mpr_status mpr_energy(mpr_ctx* ctx, double* h_e_per_bond);
/* z_min, z_max of Eq. 1 per grid, host float [batch]. */
mpr_status mpr_get_transform(mpr_ctx* ctx, float* h_zmin, float* h_zmax);
/* Fixed-site bitmask as built by mpr_create: device uint32 [batch][ceil(rows*cols/32)],
 * bit (n & 31) of word (n >> 5) = 1 for a sample site n = row*cols + col. Asynchronous. */
mpr_status mpr_get_mask_bits(mpr_ctx* ctx, uint32_t* d_bits);
/* Per-grid statistics, host mpr_stats [batch]. Synchronises. */
mpr_status mpr_get_stats(mpr_ctx* ctx, mpr_stats* h_out);
/* Number of kernels this context has launched so far (bench bookkeeping). */
mpr_status mpr_get_launch_count(mpr_ctx* ctx, uint64_t* h_count);
/* Temporal blocking of the sweep kernel: one launch advances every tile by up to
 * `k` whole sweeps of Alg. 1 on a shared-memory copy of the tile and its halo.  The result does not depend
 * on k (halo sites are recomputed bit for bit: the random numbers are keyed by site and sweep); this call
 * exists so that tests can drive every depth.  k = 0 restores the default (halo / 2; 1024 for a grid that is
 * one tile); k above the default is MPR_ERR_ARG.  Host-side only. */
mpr_status mpr_set_pass_depth(mpr_ctx* ctx, uint32_t k);
/* Schedule of mpr_simulate for a batch: `grids` > 0 runs the M x sweeps_per_real sweeps of step 6
 * for `grids` grids at a time, group after group, instead of every grid in every launch, so that a group's state can
 * stay in the L2 cache between consecutive passes (one 2048 x 2048 grid is 2 x 32 MiB of vectors).  The result does not
 * depend on the schedule (grids are independent).  0 = all grids in every launch (default).  Ignored with chains > 1.
 * Host-side only. */
mpr_status mpr_set_grid_group(mpr_ctx* ctx, int grids);
/* The tiling mpr_create chose: core tile rows x cols, halo width, and the current pass depth. */
mpr_status mpr_get_tiling(mpr_ctx* ctx, int* h_tile_rows, int* h_tile_cols, int* h_halo, uint32_t* h_pass_depth);

const char* mpr_status_string(mpr_status s);
/* Text of the last CUDA error seen by this library in the calling process. */
const char* mpr_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MPR_H */
