/* hawkes.h -- C ABI of the B200-native phylogenetic-Hawkes likelihood library.
 *
 * The library evaluates, on one NVIDIA B200 (sm_100a) in fp64, the hot path of the phylogenetic
 * Hawkes process of Holbrook, Ji & Suchard (arXiv 2103.03348; "PAPER.md" below):
 *
 *   lambda_n = sum_{n'} [ B_{nn'} + theta_{n'} k_{nn'} ]                        PAPER.md:60, 78 (Eq. 1)
 *   B_{nn'}  = mu0 tau_x^-D tau_t^-1 phi_D((x_n-x_n')/tau_x) phi_1((t_n-t_n')/tau_t) I[x_n != x_n']
 *   k_{nn'}  = xi0 omega h^-D exp(-omega (t_n-t_n')) phi_D((x_n-x_n')/h) I[t_n' < t_n]
 *   ell      = sum_n log lambda_n - Lambda(t_N)                                  PAPER.md:76 (Eq. 1)
 *   Lambda   = mu0 sum_n [Phi((t_N-t_n)/tau_t) - Phi(-t_n/tau_t)]
 *            + xi0 sum_n theta_n (1 - exp(-omega (t_N-t_n)))                     PAPER.md:72; Eq. 7, l.253
 *   d ell/d theta_m    = sum_{t_m<t_n} k_{nm}/lambda_n - xi0 (1 - e^{-omega (t_N-t_m)})   Eq. 4, l.137
 *   d2 ell/d theta_m^2 = - sum_{t_m<t_n} (k_{nm}/lambda_n)^2                              Eq. 5, l.143
 *
 * plus the gradient and Hessian with respect to the six hyperparameters (mu0, tau_x, tau_t, xi0, h,
 * omega) -- always in that order -- that BASELINE.json's north_star adds (the paper samples them by
 * Metropolis-Hastings; the derivative formulas are in DESIGN.md).  phi_D / Phi are the
 * standard normal pdf in D dimensions / cdf.  The time-Gaussian factor of the background
 * is north_star's (the paper's background is space-only): DESIGN.md reading R1.
 *
 * Conventions (all entry points)
 *  - Events are time-sorted: t[0] <= t[1] <= ... <= t[n-1]; t_N = t[n-1].  Ties are
 *    allowed and do not excite each other (strict '<').
 *  - x is SoA fp64: x[d*n + i] is coordinate d of event i, d < dim, dim in {1,2,3}.  theta[i] >= 0.
 *  - Unless an entry point says HOST, every data/output pointer is a DEVICE pointer to fp64 memory on
 *    the context's device, owned by the caller, and is not retained after the work queued on `stream`
 *    completes.  `p` is always a HOST pointer and is read before the call returns.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls only enqueue
 *    work; they never synchronise and never allocate.  One context serves one stream at a time.
 *  - A NULL output pointer means "not wanted".
 *  - Return value: 0 = HAWKES_OK; < 0 = error detected on the host, nothing was enqueued or written.
 *    Conditions that depend on the data (unsorted times, non-finite input, a zero rate) are detected
 *    on the device and reported by hawkes_last_status().
 *  - Results are bit-identical from run to run for identical inputs (fixed tile -> partial -> reduce
 *    order, no floating-point atomics).
 *  - Exponentials whose value is below 2^-1020 are flushed to zero (reading R15), and the
 *    indicator I[x_n != x_n'] is evaluated as |x_n - x_n'|^2 != 0 in fp64 (reading R3).
 */
#ifndef HAWKES_B200_H
#define HAWKES_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    double mu0;    /* background weight                        > 0 */
    double tau_x;  /* background spatial bandwidth             > 0 */
    double tau_t;  /* background temporal bandwidth            > 0 */
    double xi0;    /* self-excitation weight (paper: theta_0)  > 0 */
    double h;      /* self-excitation spatial bandwidth        > 0 */
    double omega;  /* self-excitation decay rate (1/time)      > 0 */
} hawkes_params;

typedef struct hawkes_ctx hawkes_ctx; /* opaque; owns device scratch memory only */

/* status codes */
enum {
    HAWKES_OK = 0,
    HAWKES_ERR_ARG = -1,         /* NULL/negative/oversized argument, n > n_max, dim mismatch     */
    HAWKES_ERR_PARAM = -2,       /* a hyperparameter is not finite and > 0                          */
    HAWKES_ERR_UNSORTED = -3,    /* device-detected: t is not non-decreasing                        */
    HAWKES_ERR_CUDA = -4,        /* a CUDA call failed (no device, launch failure, ...)             */
    HAWKES_ERR_NOMEM = -5,       /* scratch allocation failed                                       */
    HAWKES_ERR_UNSUPPORTED = -6, /* dim not in {1,2,3}; dense Hessian with n > 4096                 */
    HAWKES_ERR_NONFINITE = -7,   /* device-detected: NaN/Inf in x, t or theta, or theta < 0         */
    HAWKES_ERR_TOO_LARGE = -8,   /* hawkes_loglik_static: n exceeds HAWKES_STATIC_N_MAX             */
    HAWKES_WARN_ZERO_RATE = 1    /* device-detected: some lambda_n == 0 => ll = -inf, entries that
                                    divide by that lambda_n are NaN (always so for n == 1)          */
};

/* `want` bits of hawkes_eval */
enum {
    HAWKES_WANT_LL = 1,
    HAWKES_WANT_GRAD_THETA = 2,
    HAWKES_WANT_GRAD_HYPER = 4,
    HAWKES_WANT_HESS_THETA = 8,
    HAWKES_WANT_HESS_HYPER = 16,
    HAWKES_WANT_HESS_CROSS = 32
};

/* Create a context for problems of up to n_max events in `dim` dimensions on CUDA device `device`;
 * allocates all scratch (about 200 B per event + 60 MB) once.  *out is set only on success. */
int hawkes_create(hawkes_ctx** out, int64_t n_max, int dim, int device);
void hawkes_destroy(hawkes_ctx* ctx);
const char* hawkes_strerror(int status);

/* Synchronises `stream` and returns the data-dependent status of the most recent evaluation queued
 * on this context: 0, HAWKES_WARN_ZERO_RATE, HAWKES_ERR_UNSORTED or HAWKES_ERR_NONFINITE (errors win
 * over warnings).  When it returns an error the outputs of that evaluation are unspecified. */
int hawkes_last_status(hawkes_ctx* ctx, void* stream);

/* ell (Eq. 1).  ll: 1 double. */
int hawkes_loglik(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                  const hawkes_params* p /*HOST*/, double* ll, void* stream);

/* ell, d ell/d theta (Eq. 4; all n entries, w.r.t. theta itself) and d ell/d(mu0,tau_x,tau_t,xi0,h,omega).
 * grad_theta: n doubles; grad_hyper: 6 doubles. */
int hawkes_grad(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                const hawkes_params* p /*HOST*/, double* ll, double* grad_theta, double* grad_hyper,
                void* stream);

/* Second derivatives of ell (true sign: the theta-diagonal is <= 0; the paper's preconditioner is its
 * negative).  hess_theta_diag: n doubles, d2 ell/d theta_m^2 (Eq. 5).  hess_hyper: 36
 * doubles, row-major symmetric 6x6.  hess_cross: n*6 doubles row-major, d2 ell/d theta_m d p. */
int hawkes_hessian(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                   const hawkes_params* p /*HOST*/, double* hess_theta_diag, double* hess_hyper,
                   double* hess_cross, void* stream);

/* One fused evaluation sharing the two pairwise passes across all requested outputs (what an HMC
 * leapfrog step and the benchmark call).  `want` selects outputs; a wanted output whose pointer is
 * NULL is HAWKES_ERR_ARG.  Outputs not selected are not touched. */
int hawkes_eval(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                const hawkes_params* p /*HOST*/, uint32_t want, double* ll, double* grad_theta,
                double* grad_hyper, double* hess_theta_diag, double* hess_hyper, double* hess_cross,
                void* stream);

/* The same evaluation with HOST buffers on both sides (pinned or pageable): copies x, t, theta to the
 * device, evaluates, copies the selected outputs back, all on `stream`, and synchronises `stream`
 * before returning.  Returns the host status or, if that is 0, the device status of the evaluation. */
int hawkes_eval_host(hawkes_ctx* ctx, int64_t n, const double* x /*HOST*/, const double* t /*HOST*/,
                     const double* theta /*HOST*/, const hawkes_params* p /*HOST*/, uint32_t want,
                     double* ll /*HOST*/, double* grad_theta /*HOST*/, double* grad_hyper /*HOST*/,
                     double* hess_theta_diag /*HOST*/, double* hess_hyper /*HOST*/,
                     double* hess_cross /*HOST*/, void* stream);

/* Correctness-only, n <= 4096: the dense block d2 ell/d theta_m d theta_m' = - sum_n k_nm k_nm' /
 * lambda_n^2 (Lambda is linear in theta), row-major n*n doubles.  Uses n*n*8 bytes of caller memory
 * only (hess_theta itself is the scratch). */
int hawkes_hessian_theta_dense(hawkes_ctx* ctx, int64_t n, const double* x, const double* t,
                               const double* theta, const hawkes_params* p /*HOST*/,
                               double* hess_theta, void* stream);

/* ---- Log-likelihood without any device allocation -------------------------------------------------------------------
 * Every other evaluation needs a hawkes_ctx, and hawkes_create obtains its scratch with cudaMalloc.  Some programs that
 * want ell (Eq. 1, PAPER.md:76-78 -- e.g. the Metropolis-Hastings updates of the hyperparameters, which use likelihood
 * evaluations only) cannot do that: a host application whose own pool has already claimed the whole
 * device, so that a cudaMalloc from a library fails or is forbidden by its memory accounting; a sampler thread that
 * must not stall the other streams of the process (cudaMalloc / cudaFree serialise the device); a plug-in loaded
 * into a process that hands it input and output buffers and nothing else.  This one call serves them.  It needs no
 * context and calls no cudaMalloc, cudaFree or other allocating routine: the intermediates of the evaluation (packed
 * event records, pass-1 partial sums, lambda_n, block sums) live in a fixed array that is part of the library image --
 * about 9 MB of device memory on every GPU on which the library is loaded, held until the process exits -- which is why
 * the problem size is capped:
 *
 *     n <= HAWKES_STATIC_N_MAX (32,768 events; the paper's 23,422 cases fit);  larger n: HAWKES_ERR_TOO_LARGE, nothing
 *     is enqueued or written.
 *
 * It is hawkes_loglik with the ordered-pair pass 1 (the kernels are the same ones; only where their scratch lives
 * differs), for the default space-time background.  Arguments as for hawkes_loglik, all on the CURRENT device of the
 * calling thread: x [dim*n], t [n], theta [n], ll [1] DEVICE; p HOST; dim in {1,2,3}.  status_out: DEVICE, one uint32,
 * or NULL -- receives the data-dependent status of this evaluation as a bit set (HAWKES_STATIC_BIT_*; 0 = clean), the
 * counterpart of hawkes_last_status for a caller without a context; it is written on `stream` like ll.
 *
 *  - The first call on each device sets that device up: it looks up the device address of the array, raises the
 *    shared-memory limit of the pairwise kernel and copies the 2 KB exponential table into the array with a blocking
 *    cudaMemcpy.  Make that first call outside any stream capture; later calls only enqueue work on `stream`.
 *  - All calls in the process share the one array per device, and the array keeps whatever the previous call left in
 *    it.  Each call clears the status words it accumulates into and overwrites everything else before reading it, so
 *    calls that run one after the other on the GPU are independent of each other.  Two calls whose kernels can overlap
 *    on the GPU (different streams without an ordering between them, or two host threads) race on the array and give
 *    wrong results: order them.  The contexts of hawkes_create have their own scratch and are not affected. */
#define HAWKES_STATIC_N_MAX 32768
enum { HAWKES_STATIC_BIT_UNSORTED = 1, HAWKES_STATIC_BIT_NONFINITE = 2, HAWKES_STATIC_BIT_ZERO_RATE = 4 };
int hawkes_loglik_static(int64_t n, int dim, const double* x, const double* t, const double* theta,
                         const hawkes_params* p /*HOST*/, double* ll, uint32_t* status_out, void* stream);

/* Helper, not on the hot path: stable argsort of the events by time and gather into SoA outputs
 * (x_out[dim*n], t_out[n], theta_out[n]); perm[i] = input index of output event i (int64).
 * Inputs and outputs must not alias. */
int hawkes_sort_events(hawkes_ctx* ctx, int64_t n, int dim, const double* x_in, const double* t_in,
                       const double* theta_in, double* x_out, double* t_out, double* theta_out,
                       int64_t* perm, void* stream);

/* Dense theta-theta Hessian block of the sequenced events: for the m events idx[0..m),
 *   hess_block[k*m + k'] = d2 ell / d theta_idx[k] d theta_idx[k'] = - sum_n k_{n idx[k]} k_{n idx[k']} / lambda_n^2
 * (Lambda is linear in theta; the diagonal is Eq. 5), row-major m x m doubles, symmetric, DEVICE.
 * idx: DEVICE int64 [m].  Uses an n x m scratch matrix that the context allocates on first use and keeps (shared
 * with hawkes_hmc_run's kernel matrix): this call may allocate.  dim <= 2 (HAWKES_ERR_UNSUPPORTED otherwise).  Not a
 * hot-path call: a plain tiled fp64 contraction. */
int hawkes_hessian_theta_block(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                               const hawkes_params* p /*HOST*/, int64_t m, const int64_t* idx, double* hess_block,
                               void* stream);

/* Background model of the context (readings R1, R2).
 *   HAWKES_BG_SPACE_TIME (default): Gaussian-space x Gaussian-time background, the model at the top of this file.
 *   HAWKES_BG_SPACE_ONLY: the paper's background exactly as printed -- B_{nn'} = mu0 tau_x^-D phi_D((x_n-x_n')/tau_x)
 *     I[x_n != x_n'] with the integral term printed beside it, mu0 t_N.  tau_t is then
 *     unused (it must still be > 0) and every derivative with respect to it is exactly 0.
 * Applies to every later evaluation of the context.  HAWKES_ERR_ARG for another value. */
enum { HAWKES_BG_SPACE_TIME = 0, HAWKES_BG_SPACE_ONLY = 1 };
int hawkes_set_background_mode(hawkes_ctx* ctx, int mode);

/* ---- Exact-zero skipping: a separately reported variant of the evaluation ---------------------
 * A term of Eq. 1 or Eq. 4 is exp(-z) with z = |dx|^2/(2 tau_x^2) + dt^2/(2 tau_t^2)
 * (background) or z = |dx|^2/(2 h^2) + omega dt (self-excitation); in IEEE double arithmetic it is exactly +0.0 once
 * z > 745.14.  hawkes_skip_plan orders the events as the leaves of a space-time k-d tree, boxes every run of 128 of them and
 * lists the (target tile, source run) pairs whose smallest possible z is below 746 (for the self-excitation: that
 * also hold a causal pair); hawkes_eval_skip then runs the two pairwise passes over those lists only.  Nothing but
 * exact zeros is left out, so each output differs from hawkes_eval's by summation order alone (same tolerance).
 *
 * hawkes_skip_plan: x (dim x n, coordinate-major) and t (n) are HOST or DEVICE pointers; the events may be in any
 *   order (time-sorted input is not required by this variant).  Synchronous, and it allocates.  The first plan of a set
 *   of events copies them to the host once for the k-d order and the boxes (O(n log n)); the work lists (one box test
 *   per tile pair, count / scan / fill) and their cut into workers are built by kernels.  The context owns the plan
 *   until the next hawkes_skip_plan or hawkes_destroy.  The plan depends on the events, the hyperparameters and the background mode
 *   -- not on theta -- so one plan serves every evaluation of an HMC trajectory.  Planning the same events again for
 *   other hyperparameters (what an MCMC sweep does between HMC updates) keeps the order and the boxes as long as
 *   every cut-off radius stays within a factor 2 of the one the order was built for, and rebuilds only the lists: the
 *   events are recognised by a comparison on the device and are not brought to the host again.
 *   Errors: HAWKES_ERR_ARG, HAWKES_ERR_PARAM, HAWKES_ERR_NONFINITE (events), HAWKES_ERR_NOMEM, HAWKES_ERR_CUDA,
 *   HAWKES_ERR_UNSUPPORTED (work lists do not fit the context's partial buffers, or a list has 2^29 items or more).
 *   A call that fails leaves the context WITHOUT a plan: the previous plan, if there was one, has been released too
 *   (its buffers are handed to the new plan while that is being built), so hawkes_eval_skip, hawkes_posterior_z_skip
 *   and hawkes_hmc_run variants 3 / 4 return HAWKES_ERR_ARG until a later hawkes_skip_plan succeeds.
 * hawkes_eval_skip: arguments, outputs (in the caller's event order), stream semantics and device status as
 *   hawkes_eval, without the cross block (`want` bits 0..4).  HAWKES_ERR_ARG if there is no plan or it was built
 *   for another n, other hyperparameters or another background mode; the caller guarantees x and t are the planned
 *   events.  HAWKES_ERR_UNSORTED is never raised here.
 * hawkes_skip_stats: out[0..8] = pass-1 items with a live background, with a live self-excitation, of the dense
 *   pass; pass-2 items, of the dense pass; workers of pass 1, of pass 2 (item = 256 records x 128 records); items of
 *   the background evaluated once per unordered pair (levels 0 and 1; 0 if that form is not in use); 1 if this plan
 *   kept the previous plan's order and boxes (9 entries in all).
 * hawkes_skip_perm: the tree order (record i is the caller's event perm[i]) into a HOST buffer of n int64. */
int hawkes_skip_plan(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const hawkes_params* p);
int hawkes_eval_skip(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                     const hawkes_params* p, uint32_t want, double* ll, double* grad_theta, double* grad_hyper,
                     double* hess_theta_diag, double* hess_hyper, void* stream);
int hawkes_skip_stats(hawkes_ctx* ctx, int64_t* out);
int hawkes_skip_perm(hawkes_ctx* ctx, int64_t n, int64_t* perm_host);

/* Pass-1 form of the context.  Eq. 1's double sum holds the background term of
 * every ORDERED pair, and B_{nn'} = B_{n'n}:
 *   HAWKES_PASS1_AUTO (default): log-likelihood- and gradient-level evaluations compute each background exponential
 *     once per UNORDERED pair and add it to both events' sums.  This form keeps one column partial per (event, later
 *     target tile): 3072 * T * (T + 1) bytes of scratch for T = ceil(n_max / 256) tiles -- quadratic in n_max: 26 MB at
 *     n_max = 23,422, 2.9 GB at 250,000.  hawkes_create allocates it up to 16 GiB (n_max <= 605,184 events); a larger
 *     context has no such buffer and every evaluation falls back to the ordered-pair kernel, about 30 % slower at these
 *     levels (hawkes_pass1_is_symmetric tells which form a context uses);
 *   HAWKES_PASS1_DENSE: every evaluation uses the ordered-pair kernel.
 * Same sums in another order.  Applies to every later evaluation and to later hawkes_skip_plan calls.
 * hawkes_pass1_is_symmetric: 1 if an evaluation whose pass 1 runs at `level` (0: ll / theta-gradient, 1: + hyper-
 * gradient, 2: + hyper-Hessian) would take the once-per-unordered-pair form, else 0 (benchmarks label their lines
 * with it). */
enum { HAWKES_PASS1_AUTO = 0, HAWKES_PASS1_DENSE = 1 };
int hawkes_set_pass1_mode(hawkes_ctx* ctx, int mode);
int hawkes_pass1_is_symmetric(const hawkes_ctx* ctx, int level);

/* ---- One evaluation sharded across several GPUs ---------------------------------
 * One process per GPU, every rank holding all events.  The pair space of each pairwise pass (Eq. 1; Eq. 4,
 * PAPER.md:137) is cut into world x W pieces of equal modelled cost, rank r evaluating pieces [r W, (r+1) W); a rank
 * produces PARTIAL sums per event, which the caller exchanges between the phases with one all-gather per pass (the
 * binding uses torch.distributed / NCCL) and which the next phase adds in rank order:
 *
 *   hawkes_shard_pass1   (rank, world)  events -> part_out[hawkes_shard_part_doubles(n, want, 1)]: the rank's partial moment
 *                                       sums of lambda_n (background and self-excitation sums, and their r^2 / dt moments
 *                                       when hyperparameter derivatives are wanted)
 *   -- all-gather: parts_all = [world][that many doubles], rank-major --
 *   hawkes_shard_reduce1 (world)        parts_all -> lambda_n (kept by the context), ll, grad_hyper, hess_hyper.  Every rank
 *                                       runs it on the same numbers in the same order: replicated, bit-identical results.
 *   hawkes_shard_pass2   (rank, world)  -> part2_out[hawkes_shard_part_doubles(n, want, 2)]: the rank's partial c_m (and d_m)
 *   -- all-gather: parts2_all = [world][that many doubles] --
 *   hawkes_shard_finish  (world)        parts2_all -> grad_theta[n], hess_theta_diag[n] (Eq. 4, Eq. 5), replicated.
 *
 * `want`: bits LL .. HESS_HYPER of hawkes_eval (no cross block), the same in all four calls and on all ranks; x, t, theta,
 * p as for hawkes_eval; world <= 64.  All pointers DEVICE; the calls enqueue on `stream`.  hawkes_shard_reduce1 and
 * hawkes_shard_finish never synchronise or allocate.  The two pass calls do both on occasion: they cudaMalloc their partial-slot
 * buffers on first use, and when a cut needs larger ones they cudaFree the old buffer first, which waits for all work on the
 * device (the first evaluation of a given (n, want, world), in practice; later ones only enqueue).  Device
 * status as hawkes_eval (hawkes_last_status after hawkes_shard_reduce1).  With world = 1 the four calls compute what
 * hawkes_eval computes (another summation order).  Results are bit-identical run to run for a given world.
 * hawkes_shard_workers: W of the two passes for this context and `want` (diagnostics).
 * hawkes_plan_segments: HOST-only, needs no device.  The cut itself, for tests and tools: for the workers
 *   [w_begin, w_end) of a pass (1 or 2) cut into workers_total pieces at moment level `level` (0..2; `symmetric` = the
 *   once-per-unordered-pair form of pass 1) it writes up to `cap` rows (worker, tile, j_begin, j_end, partial slot) into
 *   seg[cap*5] -- worker w evaluates, for the 256 events of `tile`, the streamed events [j_begin, j_end) -- and returns
 *   the number of rows there are (call again with a larger buffer if it exceeds cap), or a negative status. */
int64_t hawkes_shard_part_doubles(int64_t n, uint32_t want, int phase);
int hawkes_shard_pass1(hawkes_ctx* ctx, int64_t n, const double* x, const double* t, const double* theta,
                       const hawkes_params* p /*HOST*/, uint32_t want, int rank, int world, double* part_out, void* stream);
int hawkes_shard_reduce1(hawkes_ctx* ctx, int64_t n, const hawkes_params* p /*HOST*/, uint32_t want, int world,
                         const double* parts_all, double* ll, double* grad_hyper, double* hess_hyper, void* stream);
int hawkes_shard_pass2(hawkes_ctx* ctx, int64_t n, const hawkes_params* p /*HOST*/, uint32_t want, int rank, int world,
                       double* part2_out, void* stream);
int hawkes_shard_finish(hawkes_ctx* ctx, int64_t n, const hawkes_params* p /*HOST*/, uint32_t want, int world,
                        const double* parts2_all, double* grad_theta, double* hess_theta_diag, void* stream);
int hawkes_shard_workers(const hawkes_ctx* ctx, uint32_t want, int* workers_pass1 /*HOST*/, int* workers_pass2 /*HOST*/);
int64_t hawkes_plan_segments(int64_t n, int pass, int level, int symmetric, int workers_total, int w_begin, int w_end,
                             int64_t* seg /*HOST*/, int64_t cap);

/* After an evaluation queued on this context has been enqueued: copies of the per-event rates
 * lambda_n (n doubles) into a caller buffer, on `stream`.  For tests and diagnostics. */
int hawkes_get_lambda(hawkes_ctx* ctx, int64_t n, double* lambda_out, void* stream);

/* Diagnostics, as hawkes_get_lambda: the per-event derivatives of lambda_n (Eq. 1) that the O(N) reduction
 * formed from the pass-1 moment sums in the most recent evaluation,
 *   d1_out[i*6 + p]  = d lambda_i / dp,            p over (mu0, tau_x, tau_t, xi0, h, omega)     (evaluations that
 *                      asked for grad_hyper, hess_hyper or hess_cross)
 *   d2_out[i*21 + k] = d2 lambda_i / dp dq, k over the upper triangle p <= q row-major            (evaluations that
 *                      asked for hess_hyper, after hawkes_row_moments_enable(ctx, 1))
 * in the record order of that evaluation (the caller's time order for hawkes_eval; the plan's order for
 * hawkes_eval_skip).  Either pointer may be NULL.  DEVICE buffers; copies on `stream`.  The second derivatives
 * take 168 bytes per event of extra scratch, which hawkes_row_moments_enable allocates (1) or frees (0):
 * that call may allocate and, when freeing, synchronises the device.  HAWKES_ERR_ARG if d2_out is wanted
 * but not enabled.  They let a test check ell, grad_hyper and hess_hyper at sizes where the O(N^2) oracle can only
 * afford a sample of rows. */
int hawkes_row_moments_enable(hawkes_ctx* ctx, int enable);
int hawkes_get_row_moments(hawkes_ctx* ctx, int64_t n, double* d1_out, double* d2_out, void* stream);

/* Debug builds only (`python -m paper_2103_03348_b200.build --guard`, loaded when HAWKES_B200_GUARD=1 is set for the
 * binding): every scratch buffer of the context lies between two 4 KB bands of a known byte pattern; this call
 * synchronises the device and returns the number of band bytes that no longer hold it (0 = no out-of-bounds write so
 * far).  HAWKES_ERR_UNSUPPORTED in the normal build (no bands).  The pool's stand-in for compute-sanitizer memcheck. */
int64_t hawkes_debug_guard_check(hawkes_ctx* ctx);

/* Launch bookkeeping for benchmarks: number of kernels this context has run since creation (kernels replayed from a
 * CUDA graph included), and the number of graph launches among the host's launch calls (hawkes_hmc_run). */
int64_t hawkes_launch_count(const hawkes_ctx* ctx);
int64_t hawkes_graph_launch_count(const hawkes_ctx* ctx);

/* Per-kernel device timing for benchmarks.  While enabled, every evaluation queued on the context
 * records CUDA events on its stream around pass 1, pass 2 (a4) and the whole
 * evaluation; a ring keeps the most recent 256 evaluations.  hawkes_profile_read() waits for those
 * evaluations, writes out[0] = number of evaluations summed, out[1] = total pass-1 milliseconds,
 * out[2] = total pass-2 milliseconds, out[3] = total milliseconds from the first to the last kernel
 * of the evaluation, out[4] = total milliseconds of step a0 (prep), out[5] = of the O(N) kernels between the
 * two passes (a2 + a3 + scalars, with their launch gaps), out[6] = of those after pass 2 (a5)
 * (out: 7 doubles, HOST), and resets the ring.  Enabling/disabling also resets it. */
int hawkes_profile_enable(hawkes_ctx* ctx, int enable);
int hawkes_profile_read(hawkes_ctx* ctx, double* out /*HOST*/);

/* Measures the fp64 FMA issue peak of the device with a register-resident DFMA-chain kernel run for
 * about `millis` milliseconds on `stream`; returns DFMA TFLOP/s (2 flops per FMA) in *tflops.
 * Synchronises.  Used by bench.py for the measured roofline denominator. */
int hawkes_fp64_peak(hawkes_ctx* ctx, double millis, double* tflops /*HOST*/, void* stream);

/* ------------------------------------------------------------------------------------------------------
 * Phylogenetic Brownian-diffusion prior on the log-rates and the z-parametrisation of the rates
 * (BASELINE.json configs[2]).
 *
 *   theta_n = exp(z_n + beta f(t_n)) for n in the sequenced set M, theta_n = 1 otherwise; f(t) = t
 *                                                                             PAPER.md:97, 202
 *   p(z | V_G, sigma^2, tau0) = (2 pi sigma^2)^(-M/2) |V_G|^(-1/2) exp(-z^T V_G^-1 z / (2 sigma^2))   Eq. 2, l.101
 *   V_G: v_mm = tau0 + d_F(root, tip m);  v_nm = tau0 + d_F(root, MRCA(tip n, tip m))
 *
 * evaluated in O(M) by post-order message passing on the tree (PAPER.md:121 cites the algorithm; DESIGN.md
 * section 11 states the recursion used), never forming V_G.
 *
 * Tree encoding: M tips, 2M-1 nodes.  Nodes 0..M-1 are the tips, tip i carrying z[i]; nodes M..2M-2 are the
 * internal nodes in any order; parent[v] is the parent of node v, parent[root] = -1; branch[v] >= 0 is the edge
 * weight w_v between v and its parent (branch[root] is ignored).  Every internal node has exactly two children.
 */
typedef struct hawkes_tree hawkes_tree; /* opaque; owns the device copy of the tree and its scratch */

/* Validates the tree (HAWKES_ERR_ARG if it is not a rooted binary tree over tips 0..M-1 or a branch is negative
 * or non-finite), orders its internal nodes by level and uploads it.  parent, branch: HOST, 2*n_tips-1 entries.
 * Allocates; synchronises. */
int hawkes_tree_create(hawkes_tree** out, int32_t n_tips, const int32_t* parent /*HOST*/,
                       const double* branch /*HOST*/, int device);
void hawkes_tree_destroy(hawkes_tree* tree);

/* log p(z | V_G, sigma2, tau0) (Eq. 2) into *logp and d log p / d z into grad_z[M] (either may be NULL, not both).
 * z, logp, grad_z: DEVICE.  sigma2 > 0, tau0 >= 0 (HAWKES_ERR_PARAM otherwise).  One kernel on `stream`; no sync.
 * A tree whose V_G is singular (tau0 = 0 with a zero-length path) yields non-finite results, not an error. */
int hawkes_tree_prior(hawkes_tree* tree, const double* z, double sigma2, double tau0, double* logp,
                      double* grad_z, void* stream);
/* diag(V_G^-1) / sigma2 = -d2 log p / d z_m^2, the prior's own diagonal curvature, into prec_diag[M] (DEVICE), in
 * O(M) by an upward and a downward sweep over the message variances.  Uses the tree's global scratch: do not run
 * it concurrently with hawkes_tree_prior on another stream. */
int hawkes_tree_precision_diag(hawkes_tree* tree, double sigma2, double tau0, double* prec_diag, void* stream);
int32_t hawkes_tree_levels(const hawkes_tree* tree);        /* depth of the level schedule (diagnostics) */
int64_t hawkes_tree_launch_count(const hawkes_tree* tree);  /* kernels launched since creation */

/* theta[i] = 1 for every i < n, then theta[idx[k]] = exp(z[k] + beta * t[idx[k]]) for k < m.
 * idx: DEVICE int64 [m], distinct, each in [0, n).  z [m], t [n], theta [n]: DEVICE. */
int hawkes_theta_from_z(hawkes_ctx* ctx, int64_t n, int64_t m, const int64_t* idx, const double* z, double beta,
                        const double* t, double* theta, void* stream);

/* Chain rule through theta(z) for the sequenced events k < m, i = idx[k]:
 *   grad_z[k] = theta[i] grad_theta[i]                       (+ prior_grad_z[k] when that pointer is not NULL)
 *   hess_z[k] = theta[i]^2 hess_theta_diag[i] + theta[i] grad_theta[i]      (likelihood part of d2/dz_k^2)
 *   *grad_beta = sum_k t[i] theta[i] grad_theta[i]            (fixed-order sum; f(t) = t)
 * hess_theta_diag/hess_z and grad_beta are optional (NULL).  All pointers DEVICE. */
int hawkes_z_chain(hawkes_ctx* ctx, int64_t n, int64_t m, const int64_t* idx, const double* theta,
                   const double* t, const double* grad_theta, const double* hess_theta_diag,
                   const double* prior_grad_z, double* grad_z, double* hess_z, double* grad_beta, void* stream);

/* One fused evaluation of the z-posterior that HMC integrates and that configs[2] times:
 *   theta(z) -> log-likelihood, d/dtheta (and the theta-Hessian diagonal if hess_z != NULL) -> tree prior ->
 *   chain rule.  out3[0] = ell, out3[1] = log p(z | V_G, sigma2, tau0), out3[2] = their sum;
 *   grad_z[m] = d(ell + log p)/dz;  hess_z[m] = likelihood part of the diagonal second derivative (see
 *   hawkes_z_chain; the prior's Hessian -V_G^-1/sigma2 is not added).  out3, grad_z, hess_z: DEVICE, each optional.
 * Uses context scratch for theta and the theta-derivatives; enqueues only.  Only the m sequenced events have a free rate, so
 * when 2 m <= n the second pairwise pass (Eq. 4 / Eq. 5) visits the pairs (target, source idx[k]) alone -- the O(NM) cost the
 * paper states for the gradient (Alg. 2 step 2) instead of O(N^2 / 2); idx may be in any order.
 * hawkes_hmc_run's recompute variants (cache_background 0 and 1) evaluate the posterior the same way. */
int hawkes_posterior_z(hawkes_ctx* ctx, hawkes_tree* tree, int64_t n, const double* x, const double* t, int64_t m,
                       const int64_t* idx, const double* z, double beta, const hawkes_params* p /*HOST*/,
                       double sigma2, double tau0, double* out3, double* grad_z, double* hess_z, void* stream);

/* hawkes_posterior_z with the likelihood evaluated by hawkes_eval_skip (the caller has called hawkes_skip_plan for
 * these events and hyperparameters; HAWKES_ERR_ARG otherwise).  Same outputs up to summation order. */
int hawkes_posterior_z_skip(hawkes_ctx* ctx, hawkes_tree* tree, int64_t n, const double* x, const double* t,
                            int64_t m, const int64_t* idx, const double* z, double beta,
                            const hawkes_params* p /*HOST*/, double sigma2, double tau0, double* out3, double* grad_z,
                            double* hess_z, void* stream);

/* ------------------------------------------------------------------------------------------------------
 * Preconditioned HMC update of the log-rates z with all likelihood work on the GPU (
 * BASELINE.json configs[3]).  Target: log pi(z) = ell(theta(z)) + log p(z | V_G, sigma2, tau0).
 *
 *   H(z, p) = -log pi(z) + 1/2 p^T M^-1 p, M diagonal
 *   per iteration: p = sqrt(M) * normals[it];  leapfrog: p += eps/2 grad; n_leapfrog times { z += eps M^-1 p;
 *   p += eps grad } with the last kick eps/2 (the printed 1/2 in dz/dt is a typo, R7);
 *   accept iff log(uniforms[it]) < H_old - H_new and H_new is finite.
 *   Preconditioner (R6): at the start of every iteration it with
 *   it % precond_every == 0, h_m = max(-d2 ell/dz_m^2, mass_floor) is evaluated at the current state and folded
 *   into the running average  mass += (h - mass) / (number of refreshes so far, this one included).
 *   The mass matrix of the dynamics is M = mass + prior_prec, prior_prec = the constant diagonal curvature of the
 *   prior (hawkes_tree_precision_diag) or NULL for M = mass (reading R20: without it the dynamics are
 *   unstable on trees with very short branches).
 *
 * The random numbers are inputs.  The work runs on a stream of the context that is forked from `stream` when the call
 * starts and joined to it before the call returns (work queued on `stream` before / after the call is ordered before /
 * after it, as for every other entry point); the accept decision is taken on the device, the call never synchronises
 * (variant 5 excepted, see below).  It instantiates up to two CUDA graphs per call (which allocates driver memory; none when every
 * kind of iteration runs fewer than 3 times, e.g. n_iter = 1).  n_leapfrog posterior evaluations per iteration (the gradient at the current state
 * is carried over), plus one Hessian-level evaluation per refresh and one evaluation before the first iteration.
 */
typedef struct {
    int32_t n_iter;          /* iterations to run, >= 1 */
    int32_t n_leapfrog;      /* leapfrog steps per iteration, >= 1 */
    int32_t precond_every;   /* refresh interval in iterations; 0 = keep `mass` as given */
    int32_t n_refresh_done;  /* refreshes already averaged into `mass` (0 for a fresh chain) */
    double step;             /* eps > 0 */
    double mass_floor;       /* > 0 */
    int32_t cache_background; /* 0: every evaluation recomputes every pair (the paper's method).
                                 1: the theta-independent background sums of pass 1 are evaluated once per call and
                                    reused (same values; pass 1 then visits causal pairs only).
                                 2: cached kernel matrix: K[n][k] = k-term of (event n, sequenced event k) / (xi0-free
                                    constant), N x M doubles built once per call (allocated by the context on first use
                                    and kept: the one entry point that may allocate), plus lambda0 = everything that does
                                    not involve a sequenced rate; an evaluation is then two passes over K (row sums ->
                                    lambda, column sums -> d ell/d theta): HBM-bound instead of FP64-bound.  Same sums in
                                    another order.  dim <= 2 only (HAWKES_ERR_UNSUPPORTED otherwise).  Variants 2 and 5
                                    cache every constant of the call, the prior included: log p(z) = log p(0) + 1/2 z^T G z
                                    with G = -V_G^-1/sigma2 formed once per (tree, sigma2, tau0) by the O(M) algorithm at
                                    the M unit vectors (M x M doubles kept by the tree; trees of more than ~3,100 tips
                                    keep the O(M) walk), a dense matrix-vector product per evaluation.
                                 3, 4: variants 0 and 1 with every evaluation over the work lists of hawkes_skip_plan
                                    (exact zeros left out; the caller has planned these events and hyperparameters,
                                    HAWKES_ERR_ARG otherwise).  Same sums in another order.
                                 5: variant 2 with the exact zeros of K left out: after the dense build its non-zeros
                                    (acausal pairs and pairs beyond the kernel's fp64 reach are exactly +0.0) are
                                    compressed by row and by column, in index order, and an evaluation reads those
                                    lists only.  Synchronises `stream` once per call, during this set-up (the number
                                    of non-zeros sizes the arrays, allocated on first use and kept); dim <= 2. */
    int32_t flags;           /* 0, or HAWKES_HMC_NO_GRAPH: enqueue every kernel of every iteration directly.  By default an
                                iteration (its [refresh,] momentum draw, n_leapfrog evaluations and accept test) is captured
                                once into a CUDA graph -- one for iterations with a preconditioner refresh, one for those
                                without -- and replayed: one host launch per iteration.  Same kernels, same results.  A kind of
                                iteration that this call runs fewer than 3 times is enqueued directly (capture costs more than
                                it saves), and so is everything while hawkes_profile_enable is on (the timing events must be
                                recorded per evaluation, not frozen into a graph). */
} hawkes_hmc_opts;
enum { HAWKES_HMC_NO_GRAPH = 1 };

/* z [m] in-out, mass [m] in-out, normals [n_iter*m], uniforms [n_iter], trace [n_iter*4] or NULL
 * (per iteration: log pi of the state after the iteration, H_old, H_new, accepted 0/1): all DEVICE.
 * opts: HOST.  Errors as hawkes_eval (HAWKES_ERR_ARG / HAWKES_ERR_PARAM before anything is enqueued). */
int hawkes_hmc_run(hawkes_ctx* ctx, hawkes_tree* tree, int64_t n, const double* x, const double* t, int64_t m,
                   const int64_t* idx, double* z, double beta, const hawkes_params* p /*HOST*/, double sigma2,
                   double tau0, const hawkes_hmc_opts* opts /*HOST*/, const double* normals, const double* uniforms,
                   double* mass, const double* prior_prec /*DEVICE [m] or NULL*/, double* trace, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* HAWKES_B200_H */
