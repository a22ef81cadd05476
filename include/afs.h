/*
 * afs.h -- C ABI of afs-b200: batched projected gradient descent on the Walsh-Fourier objective of
 * symmetric pseudo-Boolean constraints, hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations: P:Lnn = PAPER.md line nn of arxiv/paper_2606_06656 (section / equation beside it);
 * Gnn = the reading of that number in DESIGN.md section 2.
 *
 * Conventions
 *   Polarity       True -> -1, False -> +1 (section 2.1).  An expansion FE_C is -1 when C is satisfied and
 *                  +1 when violated; the objective is minimised and equals -m at a solution.
 *   Literals       signed 1-based int32: +(v+1) is x_v, -(v+1) is NOT x_v (relaxed value -x_v, G7).
 *   Layout         every batch array is row-major [B, n] (restart-major, variable fastest), as the caller sees it.
 *                  The library keeps its own transposed working copies.
 *   Ownership      the caller owns every array argument.  The library owns the handle and its internal workspace,
 *                  which grows to the largest (B, steps) seen and is freed by afs_problem_destroy.
 *   Memory space   stated per argument: "host" or "device".  Device pointers must belong to the device the
 *                  problem was created on.
 *   Asynchrony     afs_eval_grad*, afs_round_count*, afs_pgd_run* enqueue work on `cuda_stream` (a cudaStream_t
 *                  passed as void*, NULL = the legacy default stream) and return without synchronising; they may
 *                  (re)allocate workspace, which synchronises the device, the first time a larger B is seen.
 *                  afs_problem_create / afs_problem_destroy / afs_pgd_run_host synchronise.
 *                  One handle must not be used from two streams at once (the workspace is shared).
 *   Errors         every entry point returns an afs_status; nothing is printed, nothing throws.  Invalid input is
 *                  rejected at afs_problem_create.  There is no CPU fallback: without a CUDA device every device
 *                  entry point returns AFS_ERR_CUDA.
 *   Precision      the entry points compute in fp32.  The *_f64 twins are the fp64 verification build of the same
 *                  kernels (BASELINE.json north_star: "first-20-step PGD trajectories ... in an fp64 verification
 *                  build"); they take double arrays and are not tuned.
 */
#ifndef AFS_H
#define AFS_H

#include <stdint.h>

#if defined(__GNUC__)
#define AFS_API __attribute__((visibility("default")))
#else
#define AFS_API
#endif

/* AFS_DIAG marks exported MEASUREMENT AIDS (per-launch timing, counted flops, the FMA micro-benchmark): bench.py and the
 * tests use them; nothing on the product path calls them, and a product build may leave them out. */
#define AFS_DIAG AFS_API

#ifdef __cplusplus
extern "C" {
#endif

typedef struct afs_problem afs_problem; /* opaque; owns device copies of the bucketed CSR, tables, workspace */

typedef enum {
    AFS_OK = 0,
    AFS_ERR_INVALID_ARG = 1,  /* NULL pointer, negative size, B < 1, steps < 0, non-finite lr ...           */
    AFS_ERR_BAD_TYPE = 2,     /* constraint type outside afs_ctype                                            */
    AFS_ERR_BAD_K = 3,        /* EK/CARD: k < 0 or k > L+1;  XOR: k not in {0,1};  NAE with L < 2 (G6)        */
    AFS_ERR_BAD_LITERAL = 4,  /* literal 0 or |literal| > n_vars, empty constraint, row_ptr not monotone      */
    AFS_ERR_DUP_VAR = 5,      /* the same variable twice in one constraint (G8; P:L41 assumes distinct)       */
    AFS_ERR_ALLOC = 6,        /* host or device allocation failed                                             */
    AFS_ERR_CUDA = 7,         /* CUDA runtime error, or no CUDA device                                        */
    AFS_ERR_UNSUPPORTED = 8,  /* valid request outside what this build supports (see each entry point)        */
    AFS_ERR_STATIC_LIMIT = 9  /* afs_round_count_static: n and B need more than AFS_STATIC_SCRATCH_BYTES of scratch    */
} afs_status;

/* Symmetric constraint family of P:L60 (section 2.2) plus clauses (eq. 4). */
typedef enum {
    AFS_OR = 0,   /* at least one literal true                                   */
    AFS_XOR = 1,  /* number of true literals has parity k (1 = odd, G2)          */
    AFS_AMO = 2,  /* at most one                                                  */
    AFS_EO = 3,   /* exactly one                                                  */
    AFS_EK = 4,   /* exactly k                                                    */
    AFS_NAE = 5,  /* not all equal (0 < #true < L), L >= 2                        */
    AFS_CARD = 6  /* at least k (k = 0: always true, k = L+1: never true; G5)     */
} afs_ctype;

/*
 * afs_problem_create -- S0 of the path: validate, bucket by (type, length class), build the forward and the
 * transposed CSR, upload (P:L60 problem statement; "incurred once").  Synchronous.
 *   n_vars, n_cons   n >= 1, m >= 0
 *   row_ptr  host    int64[n_cons+1], row_ptr[0] = 0, non-decreasing; constraint c owns lits[row_ptr[c]..row_ptr[c+1])
 *   lits     host    int32[nnz] signed 1-based literals, distinct variables within a constraint
 *   types    host    int32[n_cons], afs_ctype values
 *   k        host    int32[n_cons]; EK: exactly k; CARD: at least k; XOR: required parity (1 = odd); otherwise ignored
 *   device           CUDA device ordinal
 *   out              receives the handle (NULL on error)
 * Limits of this build: EK / CARD up to L = 1144 literals, otherwise AFS_ERR_UNSUPPORTED; the other types have no
 * length limit.
 */
AFS_API afs_status afs_problem_create(int32_t n_vars, int32_t n_cons, const int64_t* row_ptr, const int32_t* lits,
                              const int32_t* types, const int32_t* k, int32_t device, afs_problem** out);

/*
 * afs_problem_create_w -- afs_problem_create with per-constraint weights w_k of eq. (5):
 * F_w(X) = sum_k w_k FE_{C_k}(X)  ("adaptive constraint weighting", P:L188 (i); reading G25).  weights: host
 * float[n_cons], finite (NULL = all 1).  Objective and gradient of afs_eval_grad* / afs_pgd_run* carry the weights;
 * rounding and satisfied counts do not.  A duplicated constraint equals weight 2.  Re-weighting means
 * creating a new handle (S0 is host-side and untimed).  Short clauses with w != 1 are evaluated by the
 * materialising kernels instead of the pull formulation.
 */
AFS_API afs_status afs_problem_create_w(int32_t n_vars, int32_t n_cons, const int64_t* row_ptr, const int32_t* lits,
                                        const int32_t* types, const int32_t* k, const float* weights, int32_t device,
                                        afs_problem** out);

/* Frees the handle, its device tables and workspace.  NULL is a no-op.  Synchronises the device. */
AFS_API void afs_problem_destroy(afs_problem* p);

/*
 * afs_coeffs -- the n+1 distinct Fourier coefficients a_0..a_L of one symmetric constraint (eq. 3, P:L49-L52;
 * Appendix A closed forms P:L223-L255 with readings G2-G5).  Host only, exact big-integer numerators, result
 * within 2 ulp of the exact rational.  a_out: host double[L+1].  1 <= L <= 4096.
 * The kernels do not consume these numbers: they evaluate the same polynomial in the count basis (G10).
 */
AFS_API afs_status afs_coeffs(int32_t type, int32_t L, int32_t k, double* a_out);

/*
 * afs_eval_grad -- S1..S6: objective F[b] = sum_k FE_{C_k}(X_b) (eq. 5) and its gradient.
 *   X  device float[B,n] (read only)      F  device float[B] or NULL      G  device float[B,n] or NULL
 * G[b,v] = sum over the literals of v of sigma * dFE/dy, accumulated in a fixed order (deterministic, no float
 * atomics).  Leave-one-out gradients use prefix/suffix products or stable-direction recurrences: no division by
 * a factor that can vanish at x = +-1.
 */
AFS_API afs_status afs_eval_grad(afs_problem* p, const float* X, int32_t B, float* F, float* G, void* cuda_stream);
AFS_API afs_status afs_eval_grad_f64(afs_problem* p, const double* X, int32_t B, double* F, double* G, void* cuda_stream);

/*
 * afs_constraint_grad_l1 -- per-constraint gradient magnitudes over a batch ("adaptive constraint weighting --
 * informed by per-constraint gradient magnitudes"; reading G25):  gm[k] = sum_b sum_j |dFE_k/dy_j (X_b)|, UNWEIGHTED
 * (also on a handle created with weights), in the caller's constraint order.
 *   X  device float[B,n] (read only)      gm  device float[n_cons]
 * Fixed summation order (no float atomics).  A host loop "gm -> new weights -> afs_problem_create_w" is the adaptive
 * weighting the paper names as future work; the library provides the two device-side pieces.
 */
AFS_API afs_status afs_constraint_grad_l1(afs_problem* p, const float* X, int32_t B, float* gm, void* cuda_stream);
AFS_API afs_status afs_constraint_grad_l1_f64(afs_problem* p, const double* X, int32_t B, double* gm, void* cuda_stream);

/*
 * afs_round_count -- S9: round by sign and count satisfied constraints.  x < 0 -> True (-1); x >= 0,
 * +-0.0 and NaN -> False (+1) (G13).  Integer arithmetic, bit-exact.
 *   X  device float[B,n]     assign  device int8[B,n] or NULL (-1 True, +1 False)     sat  device int32[B]
 */
AFS_API afs_status afs_round_count(afs_problem* p, const float* X, int32_t B, int8_t* assign, int32_t* sat,
                           void* cuda_stream);
AFS_API afs_status afs_round_count_f64(afs_problem* p, const double* X, int32_t B, int8_t* assign, int32_t* sat,
                               void* cuda_stream);

/*
 * afs_round_count_static -- afs_round_count (fp32) for callers that must not allocate device memory at call time.
 *
 * Which callers: a solver loop living inside a host program whose framework already owns all of HBM through its own
 * pool allocator (a cudaMalloc there fails or makes the pool shrink), a latency-bound thread that cannot afford the
 * device-wide synchronisation cudaMalloc / cudaFree imply, or a component whose host forbids driver allocations after
 * set-up.  afs_round_count grows the handle's workspace with cudaMalloc the first time it sees a larger batch; this
 * entry point never does: it calls no cudaMalloc, no cudaFree and no allocating library routine, and leaves the
 * handle's workspace alone.  (The handle itself is created earlier, by afs_problem_create, which does allocate.)
 *
 * Its working memory -- the transposed copy of X and one counter per restart -- is a fixed array of
 * AFS_STATIC_SCRATCH_BYTES that is part of the library image: every GPU that loads the library holds that much until
 * the process exits.  A request needs  256-aligned(4 Bp) + 4 n Bp  bytes of it, Bp = B rounded up to a multiple of 32
 * (e.g. n = 5000 with B <= 832, or n = 1000 with B <= 4160); anything larger is refused with AFS_ERR_STATIC_LIMIT and
 * nothing is enqueued.
 *
 * Arguments, layouts, rounding rule and results are those of afs_round_count: X device float[B,n] (read only),
 * assign device int8[B,n] or NULL, sat device int32[B]; the results are bit-identical to afs_round_count's.
 * Work is enqueued on `cuda_stream`; the call does not synchronise.
 *
 * First call on a device: looks up the array's device address (once per device, under a lock) before enqueuing
 * anything.  Make that first call during set-up, before any stream capture is begun.
 *
 * Sharing: there is one array per GPU, shared by every handle, thread and stream in the process, and it keeps the
 * previous call's contents (the entry point clears what has to start at zero).  Two calls that overlap on the same GPU
 * -- different streams, or different handles -- race on it and give wrong counts; issue them on one stream, or order
 * them with events.
 */
#define AFS_STATIC_SCRATCH_BYTES (16u << 20)
AFS_API afs_status afs_round_count_static(afs_problem* p, const float* X, int32_t B, int8_t* assign, int32_t* sat,
                                          void* cuda_stream);

/*
 * afs_pgd_run -- S1..S10 looped `steps` times with no host round trip (P:L69 PGD; G11, G12, G14, G16):
 *   entry:  fixed coordinates (mask[v] != 0) of X are overwritten with mask[v]
 *   t = 0..steps:  round X_t, count satisfied constraints; a strictly larger count replaces the best
 *                  t < steps:  X_{t+1} = clip(X_t - lr * grad F(X_t), -1, +1) on free coordinates
 *   X            device float[B,n]   in: X_0, out: X_steps
 *   steps >= 0, lr finite
 *   mask         device int8[n] or NULL: 0 free, -1 fixed True, +1 fixed False
 *   best_assign  device int8[B,n] or NULL   rounded iterate with the largest count (earliest on ties)
 *   best_sat     device int32[B] or NULL    that count
 *   best_step    device int32[B] or NULL    the iterate index in [0, steps] it was first reached at
 */
AFS_API afs_status afs_pgd_run(afs_problem* p, float* X, int32_t B, int32_t steps, float lr, const int8_t* mask,
                       int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* cuda_stream);
AFS_API afs_status afs_pgd_run_f64(afs_problem* p, double* X, int32_t B, int32_t steps, double lr, const int8_t* mask,
                           int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* cuda_stream);

/*
 * afs_pgd_run_conv -- afs_pgd_run with per-restart convergence detection ("convergence criteria"; P:L152-L164:
 * restarts converge at different times and idling converged batch elements waste compute; reading G24):
 *   a restart STOPS after the first step t -> t+1 with max_v |X_{t+1}[v] - X_t[v]| < tol (free coordinates); its
 *   iterate stays X_{t+1} and conv_step[b] = t+1, the number of steps it took (-1: never stopped within max_steps).
 *   Every iterate a restart reaches is rounded and counted as in afs_pgd_run.  Stopped restarts are retired from the
 *   working batch and the remaining ones compacted (no work is spent on them).  tol = 0 never stops a restart: the call
 *   is afs_pgd_run and conv_step is -1 everywhere.  tol must be finite and >= 0.
 * Extra outputs (device, may be NULL) -- the per-restart quantities of the paper's Fig. 4-5 histograms:
 *   conv_step int32[B] ("steps")    final_sat int32[B] satisfied constraints of the returned X (#unsatisfied =
 *   n_cons - final_sat)    final_F float[B] objective of the returned X ("energy")
 * tol > 0 always takes the streaming path.  The fp32 entry decides |dX| < tol in fp32, the _f64 twin in fp64.
 */
AFS_API afs_status afs_pgd_run_conv(afs_problem* p, float* X, int32_t B, int32_t max_steps, float lr, const int8_t* mask,
                                    float tol, int8_t* best_assign, int32_t* best_sat, int32_t* best_step,
                                    int32_t* conv_step, int32_t* final_sat, float* final_F, void* cuda_stream);
AFS_API afs_status afs_pgd_run_conv_f64(afs_problem* p, double* X, int32_t B, int32_t max_steps, double lr,
                                        const int8_t* mask, double tol, int8_t* best_assign, int32_t* best_sat,
                                        int32_t* best_step, int32_t* conv_step, int32_t* final_sat, double* final_F,
                                        void* cuda_stream);

/*
 * afs_pgd_run_masks -- afs_pgd_run with one partial assignment PER RESTART (P:L140 partial-assignment completion;
 * P:L146, L188 (ii): the batch as an enumerator of completions / sub-solver): masks is device int8[B,n], row b fixes
 * the variables of restart b (0 free, -1 fixed True, +1 fixed False).  Everything else as afs_pgd_run.  Restart b's
 * result equals afs_pgd_run on that restart alone with mask = masks[b].  Always takes the streaming path; the fixed
 * variables sit on +-1 and are handled as boundary literals (no per-call folding of the long constraints).
 */
AFS_API afs_status afs_pgd_run_masks(afs_problem* p, float* X, int32_t B, int32_t steps, float lr, const int8_t* masks,
                                     int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* cuda_stream);
AFS_API afs_status afs_pgd_run_masks_f64(afs_problem* p, double* X, int32_t B, int32_t steps, double lr,
                                         const int8_t* masks, int8_t* best_assign, int32_t* best_sat, int32_t* best_step,
                                         void* cuda_stream);

/*
 * afs_pgd_run_host -- the same call with HOST buffers (all pointers host; pinned memory recommended): copies X
 * and mask to the device, runs afs_pgd_run, copies X, best_assign, best_sat, best_step back, synchronises.
 * This is the end-to-end entry point bench.py times ("e2e").  Output pointers may be NULL.
 */
AFS_API afs_status afs_pgd_run_host(afs_problem* p, float* X, int32_t B, int32_t steps, float lr, const int8_t* mask,
                            int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* cuda_stream);

/*
 * afs_problem_info -- integer facts about a handle, for tests and bench.py.  `what`:
 *   0 n_vars  1 n_cons  2 nnz  3 constraints on the pull path  4 on the medium path  5 on the long path
 *   6 scratch slots (literals whose gradient is materialised)  7 kernel launches enqueued by the last call
 *   8 workspace bytes currently held  9 1 if the last afs_pgd_run used the tile-resident kernel, else 0
 * Unknown `what` returns -1.
 */
AFS_API int64_t afs_problem_info(const afs_problem* p, int32_t what);

/*
 * afs_set_option -- tuning knobs (all have defaults; tests use them to force code paths).  `what`:
 *   0 execution mode of afs_pgd_run: 0 auto, 1 force the streaming (one launch per phase per step) path,
 *     2 force the tile-resident path (AFS_ERR_UNSUPPORTED at run time if the instance does not fit)
 *   1 per-launch timing stride (see afs_profile_read); 0 = off
 *   2 streaming path: every `value` PGD iterations the restarts whose iterate did not change in the last step (a fixed
 *     point of the deterministic PGD map: they can never move again) are retired with their final results and the
 *     remaining ones compacted, so that later iterations work on the active restarts only.  Results are
 *     bit-identical to value = 0 (never), which tests use as the reference.  Default 32.
 * Returns AFS_ERR_INVALID_ARG for unknown options or values.
 */
AFS_API afs_status afs_set_option(afs_problem* p, int32_t what, int64_t value);

/*
 * Per-launch device timing, for bench.py's roofline of the dominant kernel.  afs_set_option(p, 1, stride) with
 * stride >= 1 makes afs_pgd_run* bracket every launch of each stride-th PGD iteration (and the single launch of the
 * tile-resident kernel) with CUDA events on the caller's stream; stride = 0 (default) switches it off.
 * afs_profile_read waits for the last recorded event, adds the elapsed milliseconds and launch counts of the most
 * recent afs_pgd_run* call per kernel class into ms[0..n) / launches[0..n) (host arrays, n <= AFS_KERNEL_CLASSES;
 * the caller zeroes them), and forgets the spans.  Classes:
 *   0 tile-resident PGD kernel      1 variable pass (pull gradients + S6 + S7 + S8)    2 pull-clause counts (S9)
 *   3 EK/CARD with L <= 64          4 medium class (prefix x suffix bodies; 5..8 unused)
 *   9..17 long-constraint kernel, 1..9 rows of 128 pmf cells                              18 boundary (layout changes,
 *   final count, fills)
 */
#define AFS_KERNEL_CLASSES 19
AFS_DIAG afs_status afs_profile_read(afs_problem* p, double* ms, int64_t* launches, int32_t n);

/*
 * afs_profile_flops -- after afs_profile_read: adds to flops[0..n) (host, caller-zeroed) the STATE-DEPENDENT
 * algorithmic flops the timed launches of each class had to do, as counted by the kernels themselves, and forgets
 * them.  Only the long-constraint kernels (classes 9..17) count: per (constraint, restart) 6 Leff Keff, the survey's
 * figure evaluated on the Leff literals that are strictly inside the cube at that iterate, with the
 * threshold left after the boundary literals that are true; 0 where the expansion is constant there.  Literals on the
 * boundary (clipped iterates, fixed variables) are exact shifts of the pmf and cost no arithmetic, so
 * the state-independent 6 L K over-counts what these kernels have to do.  Other classes add nothing.
 */
AFS_DIAG afs_status afs_profile_flops(afs_problem* p, double* flops, int32_t n);

/*
 * afs_fp32_fma_peak -- measures the plain-FP32 FMA throughput of `device` (TFLOP/s, FMA = 2 flops) with a hand-written
 * micro-benchmark kernel (independent FFMA chains on every SM, best of 5 launches, CUDA events).  Not on the product
 * path: bench.py uses it as the denominator of its "alu" roofline.  Synchronous; restores the caller's
 * current device.
 */
AFS_DIAG afs_status afs_fp32_fma_peak(int32_t device, double* tflops);

/* Static, never NULL. */
AFS_API const char* afs_status_string(afs_status s);

/* Text of the most recent CUDA runtime failure seen by the calling thread ("" if none): the CUDA error string and
 * the source location inside the library.  Diagnostic only; valid until the next failing call on this thread. */
AFS_API const char* afs_last_error_message(void);

/* ABI version of this header: bumped when a signature changes. */
AFS_API int32_t afs_abi_version(void);
#define AFS_ABI_VERSION 1

#ifdef __cplusplus
}
#endif
#endif /* AFS_H */
