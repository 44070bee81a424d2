/*
 * afsat.h -- C ABI of the B200-native AFSAT hot path (arxiv/paper_2606_06641).
 *
 * The library evaluates, for B candidate assignments X in [-1,1]^n at once, the Walsh-Fourier
 * objective  F(X) = sum_k FE_{C_k}(X)  (Eq. (2)) and its gradient over a heterogeneous
 * set of symmetric pseudo-Boolean constraints (Table 1 :87-97), fused with the projected
 * gradient step, sign rounding and the exact discrete satisfied-constraint count of Alg. 1
 * (PAPER.md:109-131).  Each FE is computed the way PAPER.md:59-67 (§2.1.2) describes: the
 * generating polynomial prod_i (1 + w^l y_i) is evaluated at DFT points w^l, w = exp(2 pi i/(k+1)),
 * and contracted with a precomputed coefficient vector built with the tailored, conjugate-symmetric
 * DFT and deferred division of PAPER.md:141-147 (§3.5.1).  DESIGN.md states every reading.
 *
 * Conventions
 *   - True <-> -1, False <-> +1.  Literal value y_i = lit_sign_i * x_{lit_var_i};
 *     a literal is true iff y_i < 0.  A variable rounds to True iff x < 0 (x = 0, -0.0 -> False).
 *   - X and G are VARIABLE-MAJOR, candidate-minor:  x[v * ldb + b],  0 <= v < n, 0 <= b < B <= ldb,
 *     ldb % 32 == 0, base pointer 128-byte aligned.  Element type is float (dtype 32) or double
 *     (dtype 64), fixed per context.  Columns b >= B are padding: never read as candidates,
 *     G padding is written as 0, X padding is left untouched.
 *   - Pointers named d_* are DEVICE pointers owned by the caller (e.g. torch tensors on the
 *     context's device); pointers named h_* are HOST pointers.  `stream` is a cudaStream_t passed
 *     as void* (NULL = the legacy default stream).  All d_* entry points are asynchronous on
 *     `stream`; the caller synchronises.  The context owns only its internal tables/workspace.
 *   - Every call returns AFSAT_OK (0) or a negative AFSAT_E_* code; no exceptions, no aborts.
 *     afsat_last_error() returns a human-readable message for the last failing call.
 *   - There is no CPU fallback: without a usable CUDA device afsat_create fails with AFSAT_E_CUDA.
 */
#ifndef AFSAT_H
#define AFSAT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct afsat_ctx afsat_ctx;

/* Constraint types: PB forms of PAPER.md Table 1 (:87-97), identifiers of Table 2 (:252-262).
 * tau = number of true literals among the k literals of the constraint.                        */
enum afsat_type {
    AFSAT_OR      = 0,  /* tau >= 1                                   param ignored          */
    AFSAT_XOR     = 1,  /* tau mod 2 == param (1 = odd = the paper's XOR, 0 = even parity)     */
    AFSAT_ATLEAST = 2,  /* tau >= param    (CARD >=; '>' t is ATLEAST t+1)       */
    AFSAT_ATMOST  = 3,  /* tau <= param    (CARD '<' t is ATMOST t-1;  AMO = ATMOST 1)         */
    AFSAT_EXACTLY = 4,  /* tau == param    (EK;  EO = EXACTLY 1)                               */
    AFSAT_NAE     = 5   /* 0 < tau < k                                param ignored          */
};

enum afsat_error {
    AFSAT_OK            =  0,
    AFSAT_E_INVALID     = -1,  /* NULL pointer, bad size / dtype / ldb / alignment, unknown type  */
    AFSAT_E_LENGTH      = -2,  /* a constraint has k < 1 or k > AFSAT_MAX_LEN                     */
    AFSAT_E_VARIABLE    = -3,  /* literal variable index outside [0, n_vars)                      */
    AFSAT_E_SIGN        = -4,  /* lit_sign not +1 / -1, or fixed[] not in {-1, 0, +1}             */
    AFSAT_E_DUPLICATE   = -5,  /* the same variable twice in one constraint (FE is multilinear)   */
    AFSAT_E_PARAM       = -6,  /* ATLEAST/ATMOST/EXACTLY with param < 0 or > k; XOR param not 0/1 */
    AFSAT_E_NOMEM       = -7,
    AFSAT_E_CUDA        = -8,  /* no device / CUDA runtime error (text in afsat_last_error)       */
    AFSAT_E_UNSAT       = -9   /* afsat_parse: the file is unsatisfiable on its face (contradictory
                                  unit assignments, a threshold no assignment can meet)           */
};

#define AFSAT_MAX_LEN 64       /* the paper's practical ceiling is ~50 literals    */

/* afsat_create flags: which host tables a signature gets (same kernels either way).
 *   paper tables : prod_i (1 + w^l y_i)/2 contracted with the tailored DFT of the integer Fourier coefficients
 *                  (PAPER.md:59-67, :141-147).  Its weights reach 2^k/N, so fp32 loses the north_star's 1e-4 on
 *                  gradients beyond k ~ 20 (the floating-point ceiling of PAPER.md:135-139).
 *   robust tables: prod_i ((1 + w^l)/2 + y_i (1 - w^l)/2) contracted with the DFT of the truth table itself
 *                  (reading B4): every factor has modulus <= 1, same FE, holds 1e-4 in fp32 up to k = 64.
 * AFSAT_FLAG_DEFAULT (automatic, SURVEY.md §8(f) NEXT #3 "per-bucket choice"): the paper tables for lengths k <= 20 and
 * the robust tables for k > 20, in both precisions -- at corner points (where projected gradient descent parks variables)
 * the paper's product form loses 1e-4 in fp32 and 1e-10 in fp64 beyond k ~ 20-25.
 * AFSAT_FLAG_ROBUST: robust tables for every signature.  AFSAT_FLAG_PAPER: paper tables for every signature
 * (the comparison mode BASELINE.json configs[3] "report deviation" asks for).  Lengths are those AFTER the
 * partial assignment has been substituted (see afsat_create).                                                  */
#define AFSAT_FLAG_DEFAULT      0u
#define AFSAT_FLAG_ROBUST       1u
#define AFSAT_FLAG_PAPER        2u

/*
 * afsat_create -- build a context for one instance.
 *   row_ptr[m+1], lit_var[nnz], lit_sign[nnz], type[m], param[m], fixed[n] (or NULL) are HOST
 *   arrays in CSR form, borrowed for the duration of the call only (copied).
 *   fixed[v]: 0 = free, -1 = fixed True (x = -1), +1 = fixed False (x = +1): the partial
 *   assignment of PAPER.md:105-107; fixed variables use that value whatever X holds, receive zero
 *   gradient and are never updated.
 *   batch = B >= 1, ldb >= B with ldb % 32 == 0, dtype = 32 or 64, device = CUDA ordinal.
 * Validates everything (see afsat_error); SUBSTITUTES the partial assignment into the constraints (PAPER.md:133:
 * a symmetric constraint restricted by fixed literals is again symmetric -- with f_T fixed-true literals its truth
 * table is the original one shifted by f_T on the remaining literals; constraints it decides outright become
 * constants of F and of the satisfied count); groups the resulting constraints by signature (length, truth table);
 * precomputes per signature the exact integer coefficients, the conjugate-symmetric root table and the contracted
 * weights (division deferred to the end); uploads the tables.
 * Validation happens before the device is touched, so invalid input is reported even without a GPU.
 */
int afsat_create(afsat_ctx **out, int32_t n_vars, int32_t n_cons, const int64_t *row_ptr,
                 const int32_t *lit_var, const int8_t *lit_sign, const uint8_t *type,
                 const int32_t *param, const int8_t *fixed, int32_t batch, int64_t ldb,
                 int32_t dtype, int32_t device, uint32_t flags);

/*
 * afsat_create_ex -- afsat_create with explicit options (every field 0 = the automatic choice).
 *   n_groups > 1: SEVERAL partial assignments ("AFSAT evenly divides up a given batch of candidate
 *     assignment amongst multiple partial assignment"): fixed is then [n_groups][n_vars] and candidates
 *     [g B / n_groups, (g + 1) B / n_groups) run under mask g.  Requires batch % (32 n_groups) == 0.
 *   tile_w: width of the candidate tiles of a step (a multiple of 32); l2_budget_bytes: bytes of L2
 *     the X and G tiles may take when the library picks the width itself (default: 13/16 of the device's L2).
 *   step_path: AFSAT_STEP_AUTO, or force AFSAT_STEP_LAUNCHES / AFSAT_STEP_PERSISTENT / AFSAT_STEP_GRAPH for afsat_step
 *     (PERSISTENT is refused with AFSAT_E_INVALID when the instance does not fit: every length <= 8, one group,
 *     X and G of one candidate in shared memory).
 */
enum afsat_step_path {
    AFSAT_STEP_AUTO = 0,
    AFSAT_STEP_LAUNCHES = 1,    /* one set of launches per iteration and candidate tile                               */
    AFSAT_STEP_PERSISTENT = 2,  /* the whole n_steps loop in ONE launch: a CTA per candidate, a thread per constraint, X and
                                   G in shared memory (small instances)                                               */
    AFSAT_STEP_GRAPH = 3        /* one iteration captured into a CUDA graph, replayed n_steps times                   */
};
typedef struct afsat_options {
    uint32_t struct_size;       /* sizeof(afsat_options) */
    uint32_t flags;             /* AFSAT_FLAG_* */
    int32_t  n_groups;          /* 0 or 1: one partial assignment */
    int32_t  step_path;         /* enum afsat_step_path */
    int64_t  tile_w;
    int64_t  l2_budget_bytes;
} afsat_options;
int afsat_create_ex(afsat_ctx **out, int32_t n_vars, int32_t n_cons, const int64_t *row_ptr,
                    const int32_t *lit_var, const int8_t *lit_sign, const uint8_t *type,
                    const int32_t *param, const int8_t *fixed, int32_t batch, int64_t ldb,
                    int32_t dtype, int32_t device, const afsat_options *opt);

void afsat_destroy(afsat_ctx *ctx);

/* Message of the last failing call on ctx (ctx == NULL: last failing afsat_create of this thread). */
const char *afsat_last_error(const afsat_ctx *ctx);

/*
 * afsat_eval_grad -- steps a1-a5:  F[b] = sum_C FE_C(X[:,b])  and  G[v][b] = dF[b]/dx_v.
 *   d_x [n][ldb] (read), d_F [B] (written; may be NULL), d_G [n][ldb] (OVERWRITTEN, not
 *   accumulated; rows of fixed variables and padding columns are 0; may be NULL for F only).
 *   The gradient is the analytic leave-one-out product (prefix x suffix), never a division.
 *   Every d_x / d_G of this header must be 16-byte aligned (the kernels use 16-byte vector accesses; a torch
 *   tensor is 256-byte aligned); a misaligned pointer is AFSAT_E_INVALID, not a fault.
 */
int afsat_eval_grad(afsat_ctx *ctx, const void *d_x, void *d_F, void *d_G, void *stream);

/*
 * afsat_check -- steps a7-a8, integer only:  sat_count[b] = #constraints satisfied by the
 *   sign-rounded X[:,b],  is_solution[b] = (sat_count[b] == m).  Bit-exact by construction.
 */
int afsat_check(afsat_ctx *ctx, const void *d_x, int32_t *d_sat_count, uint8_t *d_is_solution,
                void *stream);

/*
 * afsat_check_static -- afsat_check for callers that cannot allocate at call time (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  Same inputs, same outputs, bit for bit; the difference is
 * where the scratch of the check lives: the sign bits [n][ldb/32] of a7 and the per-candidate accumulator [ldb] of a8
 * are placed in ONE file-scope device array of AFSAT_STATIC_SCRATCH_BYTES that the library carries (every GPU that
 * loads the library holds those bytes until the process exits), not in the context's workspace.  The call makes no
 * cudaMalloc / cudaFree and calls no allocating routine: one cudaMemsetAsync and the three kernels of the check on
 * `stream`, nothing else.
 *   Needs  ldb * 4 (rounded up to 256) + n_vars * (ldb / 32) * 4  bytes; a context that needs more is refused with
 *   AFSAT_E_NOMEM and a message that names both numbers (cfg2 of BASELINE.json, n = 5000, B = 4096, needs 2.6 MB).
 *   afsat_static_setup(device) resolves the array's device address (cudaGetSymbolAddress) once per device; call it
 *   at set-up -- in particular BEFORE starting a graph capture.  afsat_check_static calls it itself if that has
 *   not happened yet for the context's device.
 *   EVERY call on a device shares the one array, whatever the context: the array keeps the last call's contents (the
 *   entry point clears what has to start at zero), and two calls that overlap on the GPU -- different streams, or
 *   different contexts on different host threads without ordering between them -- RACE on it.  Order them on one
 *   stream or with events.  The ordinary afsat_check has no such restriction.
 */
#define AFSAT_STATIC_SCRATCH_BYTES (8u << 20)
int afsat_static_setup(int32_t device);
int afsat_check_static(afsat_ctx *ctx, const void *d_x, int32_t *d_sat_count, uint8_t *d_is_solution, void *stream);

/*
 * afsat_step -- n_steps iterations of Alg. 1 with a fixed step eta, steps
 * a1-a9 fused, no host round trip between iterations:
 *     G = grad F(X(t-1));  X(t) = clamp(X(t-1) - eta G, -1, +1) on free variables of unsolved
 *     candidates;  round;  count on X(t);  if all m satisfied: is_solution = 1,
 *     first_step = step_base + t, and the candidate is frozen (executes no-ops).
 *   X(0) itself is not checked (Alg. 1 checks after each step).
 *   d_x [n][ldb] in/out.  d_F [B] (may be NULL): F at the final X (Alg. 1's output FE(X_bar); costs one more
 *   objective-only pass).  d_F_pre [B] (may be NULL): F(X(n_steps - 1)), the objective at the point where the LAST
 *   gradient was taken -- a by-product of the fused pass (the contraction a3 of the same products: no second pass;
 *   without it the fp32 kernels for k <= 8 run their gradient-only form, some 8 % faster);
 *   a caller that steps repeatedly sees Alg. 1's FE(X(t)) one iteration late.  Not written when n_steps = 0.
 *   d_sat_count [B]: satisfied count at the final X.  d_is_solution [B], d_first_step [B] (-1 = none): if
 *   resume != 0 they are read as the state left by an earlier call (frozen candidates stay frozen), else reset.
 *   h_any_solved (may be NULL): 2 x int32 in PINNED, device-mapped host memory; [0] is set to 1
 *   and [1] to the step index as soon as the first candidate is solved (poll without syncing); both are reset
 *   ({0, -1}) ON THE STREAM at the start of the call, after earlier work of the stream.
 *   How the loop runs (afsat_query AFSAT_Q_STEP_PATH): small instances run all n_steps in ONE persistent launch;
 *   others launch per iteration, or replay one captured iteration as a CUDA graph.
 */
int afsat_step(afsat_ctx *ctx, void *d_x, double eta, int32_t n_steps, int32_t step_base,
               int32_t resume, void *d_F, void *d_F_pre, int32_t *d_sat_count, uint8_t *d_is_solution,
               int32_t *d_first_step, int32_t *h_any_solved, void *stream);

/*
 * afsat_step_ls -- Alg. 1 WITH its line search and convergence test ("eta <-
 * lineSearch(FE, grad FE, s)", :125 "if eta < delta", :103).  The paper
 * names no method; reading B5 fixes backtracking with the Armijo rule along the projection
 * arc, independently per candidate (the candidates of a batch are independent searches):
 *     G = grad F(X);  eta = s_max;
 *     repeat at most max_trials times:
 *         X' = clamp(X - eta G, -1, +1) on free variables;   D = <G, X - X'>;
 *         if F(X') <= F(X) - c1 D: accept, stop;   else eta <- beta eta;
 *         if eta < delta: the candidate has CONVERGED (d_converged = 1): it keeps X and is frozen;
 *     accepted: X <- X';  round;  count;  solved candidates are frozen as in afsat_step.
 *   A candidate that exhausts max_trials without acceptance keeps X for this step and is not flagged.
 *   Every trial costs one objective-only evaluation (a1-a3, no suffix walk) of the candidates
 *   still searching; the others are skipped warp by warp.
 *   d_x [n][ldb] in/out.  d_F [B] (may be NULL): F at the final X.  d_eta [B] (may be NULL): the step
 *   length of the last iteration (accepted, or the one that fell below delta / was rejected last).
 *   d_converged [B]; d_sat_count, d_is_solution, d_first_step, resume, step_base, h_any_solved as in
 *   afsat_step (resume != 0 also reads d_converged).  0 < beta < 1, 0 <= c1 < 1, s_max > 0,
 *   delta >= 0, max_trials >= 1; otherwise AFSAT_E_INVALID.
 *   Workspace: a full gradient and a trial copy of X ([n][ldb] each), allocated on first use.
 */
int afsat_step_ls(afsat_ctx *ctx, void *d_x, double s_max, double beta, double c1, double delta,
                  int32_t max_trials, int32_t n_steps, int32_t step_base, int32_t resume,
                  void *d_F, void *d_eta, int32_t *d_sat_count, uint8_t *d_is_solution,
                  int32_t *d_first_step, uint8_t *d_converged, int32_t *h_any_solved, void *stream);

/*
 * afsat_restart -- random re-initialisation of candidates (the compiled search is "executed
 * repeatedly with different random initialisations"; :105-107: fixed variables keep their value for every
 * candidate, the remainder is random).  For every candidate b with
 * d_keep == NULL or d_keep[b] == 0:  x[v][b] = the fixed value of v if v is fixed, else
 *     u(seed, round, v, b) = ((h >> 8) * 2^-23) - 1   in [-1, 1),   exactly representable in fp32,
 *     h1 = fmix(lo ^ (b * 0x9E3779B9));  h2 = fmix((h1 + v * 0x85EBCA6B) ^ hi);  h = fmix(h2 + round * 0xC2B2AE35),
 *     lo / hi = low / high 32 bits of seed,  fmix(h): h ^= h >> 16; h *= 0x85EBCA6B; h ^= h >> 13;
 *     h *= 0xC2B2AE35; h ^= h >> 16   (all arithmetic mod 2^32).
 * A counter-based generator: the value depends only on (seed, round, v, b), never on launch geometry, so
 * the CPU oracle reproduces it bit for bit.  Kept candidates (e.g. d_keep = is_solution) are untouched.
 */
int afsat_restart(afsat_ctx *ctx, void *d_x, const uint8_t *d_keep, uint64_t seed, uint32_t round, void *stream);

/*
 * afsat_solve -- the restart loop around afsat_step (Alg. 1): up to max_rounds rounds of
 * steps_per_round fixed-step iterations each; after a round without a solution every unsolved candidate
 * is re-initialised by afsat_restart(seed, round = r) and the next round continues the step count
 * (first_step is the global iteration index).  Stops after the first round in which some candidate is
 * solved (stop_at_first != 0) or after max_rounds.  X(0) is the caller's d_x (call afsat_restart with
 * round 0xFFFFFFFF first for a random start).  Synchronises `stream` once per round (reads one flag).
 * rounds_done (HOST, may be NULL) receives the number of rounds executed.  Outputs as in afsat_step.
 */
int afsat_solve(afsat_ctx *ctx, void *d_x, double eta, int32_t steps_per_round, int32_t max_rounds,
                uint64_t seed, int32_t stop_at_first, void *d_F, int32_t *d_sat_count,
                uint8_t *d_is_solution, int32_t *d_first_step, int32_t *rounds_done, void *stream);

/*
 * afsat_step_host -- the same as afsat_step (resume = 0, step_base = 0) for HOST buffers: copies
 * h_x [n][ldb] to the device, runs n_steps, copies X, F, F_pre, sat_count, is_solution, first_step back
 * (any output pointer may be NULL) and synchronises.  Pinned host memory makes the copies
 * asynchronous; pageable memory works too.  When the step runs tile by tile the copies are pipelined by candidate
 * tile behind the evaluation.  This is the end-to-end call bench.py times.
 */
int afsat_step_host(afsat_ctx *ctx, void *h_x, double eta, int32_t n_steps, void *h_F, void *h_F_pre,
                    int32_t *h_sat_count, uint8_t *h_is_solution, int32_t *h_first_step);

/*
 * afsat_host_tables -- HOST ONLY, no device needed: the contracted weight table of one signature,
 * as the kernels consume it.  For every retained DFT point l the row
 *     table[8*p .. 8*p+7] = { Re a, Im a, Re b, Im b, Re w, Im w, Re(w b), Im(w b) }
 * such that  FE(y) = sum_p Re( w_p * prod_i (a_p + b_p y_i) )  and
 *            dFE/dy_i = sum_p Re( w_p b_p * prod_{j != i} (a_p + b_p y_j) ).
 * Real points (Im = 0 throughout) come first.  Returns the number of rows (<= AFSAT_MAX_LEN/2+1)
 * or a negative error; table must hold 8 * (AFSAT_MAX_LEN/2 + 1) doubles; n_real (may be NULL)
 * receives the number of real rows.
 */
int afsat_host_tables(int32_t type, int32_t k, int32_t param, uint32_t flags, double *table,
                      int32_t *n_real);

/*
 * afsat_host_restrict -- HOST ONLY: what a constraint becomes under a partial assignment (the
 * substitution afsat_create applies).  A constraint (type, k, param) with f_true of its literals fixed true and
 * f_false fixed false keeps k_free = k - f_true - f_false literals and, on them, the symmetric constraint whose
 * satisfying counts are  { tau' : tau' + f_true satisfies the original }.  mask[0] / mask[1] receive that set as
 * bits 0..63 / 64..127.  Returns 0 if the restricted constraint still depends on its free literals, 1 if the
 * assignment already satisfies it, 2 if it already violates it, or a negative error.
 * afsat_host_tables_mask -- afsat_host_tables for such a (k_free, mask) signature (flags: 0 = paper tables,
 * AFSAT_FLAG_ROBUST = robust tables).
 */
int afsat_host_restrict(int32_t type, int32_t k, int32_t param, int32_t f_true, int32_t f_false, int32_t *k_free,
                        uint64_t *mask);
int afsat_host_tables_mask(int32_t k, uint64_t mask_lo, uint64_t mask_hi, uint32_t flags, double *table, int32_t *n_real);

/* afsat_query -- counters and facts about a context. */
enum afsat_query_key {
    AFSAT_Q_KERNEL_LAUNCHES = 0,  /* kernels launched by this context so far                     */
    AFSAT_Q_NUM_SIGNATURES  = 1,
    AFSAT_Q_NUM_BUCKETS     = 2,  /* distinct constraint lengths                                 */
    AFSAT_Q_NNZ             = 3,
    AFSAT_Q_WORKSPACE_BYTES = 4,
    AFSAT_Q_SM_COUNT        = 5,
    AFSAT_Q_FP_INSTR_PER_CANDIDATE = 6, /* model count of FP instructions for one eval_grad of one
                                           candidate over all constraints (DESIGN.md cost model)  */
    AFSAT_Q_PROFILED_EVAL_NS = 7,       /* afsat_set_profiling: device time of the evaluation kernels
                                           (a1-a5) since profiling was switched on, in ns;
                                           SYNCHRONISES with the recorded events                  */
    AFSAT_Q_PROFILED_EVAL_LAUNCHES = 8, /* number of evaluation-kernel launches in that time       */
    AFSAT_Q_FLOP_PER_CANDIDATE = 9,     /* model flop count, same scope as key 6; both are counted on the
                                           constraint table AFTER the partial assignment was substituted */
    AFSAT_Q_NUM_GROUPS = 10,            /* partial assignments                                     */
    AFSAT_Q_STEP_PATH = 11,             /* enum afsat_step_path actually used by afsat_step        */
    AFSAT_Q_TILE_W = 12,                /* candidate tile width of a step                          */
    AFSAT_Q_LIVE_CONSTRAINTS = 13,      /* constraints that reach a kernel (group 0)               */
    AFSAT_Q_LIVE_NNZ = 14,              /* their literals (group 0)                                */
    AFSAT_Q_DECIDED_SATISFIED = 15,     /* constraints group 0's partial assignment satisfies outright */
    AFSAT_Q_L2_BYTES = 16,              /* cudaDeviceProp::l2CacheSize                             */
    AFSAT_Q_PROFILED_UPDATE_NS = 17,    /* afsat_set_profiling: device time of the update kernels (a6, a7, a9) */
    AFSAT_Q_PROFILED_CHECK_NS = 18      /* ... and of the exact count (a8); both SYNCHRONISE like key 7 */
};
int64_t afsat_query(const afsat_ctx *ctx, int32_t key);

/*
 * afsat_set_profiling -- on != 0: bracket every evaluation-kernel launch of this context with CUDA
 * events on the launching stream (the roofline numerator of bench.py is measured this way, live,
 * inside the step); on == 0: stop.  Either call resets the accumulated time.  Costs two event
 * records per launch, so it is off by default and off in every timed headline region.
 */
int afsat_set_profiling(afsat_ctx *ctx, int32_t on);

/*
 * Problem ingestion (HOST ONLY; App. A, simplifications :300-309 A.1; SURVEY.md §8(f)
 * NEXT #2).  afsat_parse reads a DIMACS CNF file or the paper's DIMACS-like hybrid PB format from
 * memory (text[0..len), need not be NUL-terminated) and returns an opaque afsat_problem holding what
 * afsat_create consumes.  Grammar: comment lines start with 'c' or '*'; 'p cnf <vars> <constraints>';
 * a constraint is  ['h'] [<id> [<threshold>]] <lit>+ 0  with <id> in { (none): disjunction,
 * x|xor: odd parity, n|nae: not all equal, a|amo: at most one, e|eo: exactly one, k|ek <int>: exactly
 * k, d|card [<|<=|>|>=]<int>: cardinality; a bare card threshold k means >= k if k > 0, < |k| if k < 0 }.
 * A literal l is variable |l| (1-based in the file, 0-based in the arrays) and is true iff that
 * variable is True (l > 0) or False (l < 0): lit_sign = +1 / -1.
 * Simplifications applied while reading (A.1): unit disjunction / unit eo -> prefix assignment; unit amo
 * discarded; card >= 1 -> disjunction; ek 1 = eo; card >= n and ek n -> all literals assigned true;
 * card >= 0 discarded; ek 0 -> all literals assigned false.  Also (reading B6): a literal
 * repeated in a disjunction is kept once, a disjunction with l and -l is discarded, a repeated variable
 * elsewhere is AFSAT_E_DUPLICATE; at-most thresholds >= the length are discarded, at-most 0 assigns all
 * literals false; contradictory assignments and unmeetable thresholds are AFSAT_E_UNSAT.
 * n_vars = max(declared <vars>, largest variable used).  The prefix assignments come back as
 * fixed[v] in {0 free, -1 True, +1 False} (the partial-assignment mask of afsat_create).
 *   afsat_problem_sizes: stats (may be NULL) receives 5 values {constraints read, variables assigned
 *     by unit extraction, constraints discarded, declared vars, declared constraints (summed over p lines)}.
 *   afsat_problem_fill: copies into caller-owned HOST arrays row_ptr[m+1], lit_var[nnz], lit_sign[nnz],
 *     type[m], param[m], fixed[n_vars].
 *   afsat_parse_error: message of the last failing afsat_parse / afsat_parse_file on this thread.
 */
typedef struct afsat_problem afsat_problem;
#define AFSAT_PARSE_MAX_VARS 0x3FFFFFFF
int afsat_parse(const char *text, int64_t len, afsat_problem **out);
int afsat_parse_file(const char *path, afsat_problem **out);
const char *afsat_parse_error(void);
int afsat_problem_sizes(const afsat_problem *p, int32_t *n_vars, int32_t *n_cons, int64_t *nnz, int64_t *stats);
int afsat_problem_fill(const afsat_problem *p, int64_t *row_ptr, int32_t *lit_var, int8_t *lit_sign,
                       uint8_t *type, int32_t *param, int8_t *fixed);
void afsat_problem_free(afsat_problem *p);

/*
 * afsat_probe_peak -- measured rates of what the path is bound by (the roofline denominators of bench.py), timed with
 * CUDA events on `device`; SYNCHRONISES.  kind 0 = scalar FFMA, 1 = packed FFMA2 (fma.rn.f32x2), 2 = DFMA: independent
 * chains, nothing else; *tflops receives the best of 5 runs in TFLOP/s (FMA = 2 flop).  kind 3 = L2 loads (16-byte,
 * bypassing L1), 4 = L2 vector REDs (red.global.add.v4.f32), 5 = both in equal parts, over a 24 MB L2-resident buffer
 * from every SM -- the access kinds of the evaluation kernels; *tflops then receives TB/s of payload (best of 3).
 * The probe allocates its own scratch.
 */
int afsat_probe_peak(int32_t device, int32_t kind, double *tflops);

const char *afsat_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AFSAT_H */
