/*
 * sup.h -- C ABI of libsup: the superiorized simultaneous-projection iteration over hyperslabs + box,
 * hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Method: arXiv 2606.27086 ("GPU-accelerated superiorization ... with SupPy"), cited as PAPER.md:L<line>.
 * Readings of the paper where it is silent or garbled are numbered A-1 .. A-22 in DESIGN.md.
 *
 *   constraint sets   C_i = { x : lb_i <= <a_i, x> <= ub_i },  i = 0..m-1        (Eq. 1-2, L384 Eq. 20)
 *   box               lo_j <= x_j <= hi_j                                          (PAPER.md:L427 BoxProjection)
 *   weights           w_i > 0, sum_i w_i = 1;  d_i = w_i / ||a_i||^2
 *   sweep             x <- P_box( x - lambda * A^T D c(x) ),   c_i = hyperslab violation of <a_i,x>   (A-1, A-2)
 *   perturbation      x <- x + beta * v,  v = -grad f / ||grad f||,  beta = beta0 * a^l,
 *                     accepted iff f(z) <= f(x)                                   (Alg. 1)
 *
 * CONVENTIONS
 *  - Every array argument is a DEVICE pointer owned by the caller unless its comment says "host".
 *    The library BORROWS A, lb, ub, box_lo, box_hi (and D_body) for the handle's lifetime and never frees them.
 *  - The library never allocates device memory.  Everything it derives (transposed CSR, the packed (value, column)
 *    copies of A and A^T that the fp32 kernels stream, row scaling, scratch vectors, reduction partials, device-side
 *    state) lives in caller-provided WORKSPACE memory whose size comes
 *    from sup_workspace_bytes().  "persistent" workspace must stay alive until sup_destroy(); "scratch"
 *    workspace is only used during the call that takes it and may be freed once that call's stream work is done
 *    (the calls that take scratch synchronise the stream before returning).
 *  - Working precision: SUP_F32 = fp32 storage and fp32 row dot products, fp64 for every global reduction,
 *    objective value, norm and step size; SUP_F64 = everything fp64.  `val`, lb, ub, box, weights, x are arrays
 *    of the handle's dtype.  Column indices are int32, row pointers int64.  CSR must be canonical: columns
 *    strictly increasing within a row, 0 <= col < n.  +-INFINITY encodes a one-sided bound.
 *  - All work is enqueued on the cudaStream_t given at sup_create (passed as void*; NULL = default stream).
 *    Calls that return a host scalar synchronise that stream; sup_project_simultaneous / sup_block_iterative /
 *    sup_superiorize are asynchronous with respect to the host.
 *  - Errors: every call returns a sup_status; nothing throws or aborts.  Argument errors are detected before
 *    any launch.  sup_last_error() gives a text for the last failure on that handle (or of sup_create when
 *    called with NULL).  There is NO CPU fallback: without a CUDA device every call fails with SUP_ERR_CUDA.
 */
#ifndef SUP_H
#define SUP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sup_ctx* sup_handle;

typedef enum {
    SUP_OK = 0,
    SUP_ERR_INVALID_ARG = 1, /* null pointer, bad size, lambda outside [0,2], a outside (0,1) (L99), ... */
    SUP_ERR_FORMAT = 2,      /* CSR not canonical, lb > ub, lo > hi, weight <= 0 */
    SUP_ERR_WORKSPACE = 3,   /* workspace too small or misaligned (256 B) */
    SUP_ERR_CUDA = 4,        /* a CUDA runtime call or kernel failed */
    SUP_ERR_STATE = 5,       /* call needs something not set (blocks, dose matrix) */
    SUP_ERR_NONFINITE = 6    /* NaN/Inf met in a reduction */
} sup_status;

typedef enum { SUP_F32 = 0, SUP_F64 = 1 } sup_dtype;

/* objective kinds of the perturbation phase */
typedef enum {
    SUP_OBJ_NONE = 0, /* no perturbation: the basic algorithm (Eq. 10 with beta v = 0) */
    SUP_OBJ_TV2D = 1, /* isotropic total variation, Eq. 15, on x viewed as ny x nx row-major */
    SUP_OBJ_TV1D = 2, /* sum |x_{i+1} - x_i|  (A-16) */
    SUP_OBJ_DOSE = 3, /* || D_body x ||^2     (A-15; north_star) */
    SUP_OBJ_MEAN = 4, /* f_Mean = (1/N_S) sum_{i in S} (D_S x)_i, Eq. 21; D_S is the matrix given to
                         sup_set_dose_matrix (its rows are the structure's voxels) */
    SUP_OBJ_TV3D = 5  /* Eq. 15 with a third difference on x viewed as nz x ny x nx (A-27) */
} sup_objective_kind;

/* step-size exponent policy (A-10) */
typedef enum {
    SUP_STEP_PER_TRIAL = 0, /* one persistent counter l, beta = beta0*a^l used then l += 1 on EVERY trial */
    SUP_STEP_PER_SWEEP = 1  /* literal Alg. 1: beta_{k,j} = beta0 * a^(k+j), j reset at every reduction step */
} sup_step_policy;

/* step-size rule of the perturbation phase */
typedef enum {
    SUP_RULE_POWER = 0,   /* beta = beta0 * a^l, trial loop with the accept test f(z) <= f(x) (Algorithm 1) */
    SUP_RULE_ADAPTIVE = 1 /* Eq. 11: beta = 0 if f(x) <= f_ref, else (f(x) - f_ref)/||g_f(x)||; the step
                             x - ((f(x) - f_ref)/||g||^2) g is taken without a trial loop, N times per phase, l is not used
                             (N, beta0, a of the call: only N is read).  TV and dose objectives.  The update of f_ref is the
                             reading DESIGN.md A-30 (the paper only cites the rule: parity unpinned for that part) */
} sup_step_rule;

/* what a workspace query is for */
typedef enum { SUP_WS_CREATE = 0, SUP_WS_BLOCKS = 1, SUP_WS_DOSE = 2 } sup_ws_kind;

/* m x n CSR matrix in device memory */
typedef struct {
    int64_t m, n, nnz;
    const int64_t* rowptr; /* [m+1], rowptr[0] = 0, rowptr[m] = nnz */
    const int32_t* col;    /* [nnz] */
    const void* val;       /* [nnz] of the handle's dtype */
} sup_csr;

/* options of sup_superiorize; zero-initialise, then set what is needed */
typedef struct {
    int objective;         /* sup_objective_kind */
    int64_t shape[3];      /* TV2D: {ny, nx, 0} with ny*nx == n; TV3D: {nz, ny, nx} with nz*ny*nx == n; others ignored */
    double lambda;         /* relaxation in [0,2] (Eq. 3) */
    int block_iterative;   /* 0: simultaneous sweep; 1: block-iterative sweep (needs sup_set_blocks) */
    int step_policy;       /* sup_step_policy */
    int64_t ell0;          /* step-size exponent to start from (resume state) */
    int64_t k0;            /* index of the first sweep (resume state; only PER_SWEEP uses it) */
    int trace_mode;        /* 1: after every sweep also evaluate proximity (Eq. 5) and f(x) into `trace` (slow: one extra pass) */
    double* trace;         /* device, [n_iter][4] = {proximity mode 0, f(x), #trials, l} after each sweep; NULL = off */
    int8_t* decisions;     /* device, [decisions_cap]: 1 = accepted / 0 = rejected, one per trial; NULL = off */
    double* decision_f;    /* device, [decisions_cap][2] = {f(z), f(x^{k,n})} per trial; NULL = off */
    int64_t decisions_cap;
    int use_graph;         /* 1: capture one sweep into a CUDA graph and replay it (default path of bench.py) */
    int64_t n_restart;     /* > 0: restarted perturbations: at the start of sweep k = r * n_restart,
                              r = 1, 2, ..., the exponent l is reset to r (PER_TRIAL policy; A-24).  0: off */
    int algorithm;         /* sup_algorithm: the feasibility-seeking operator T of Eq. 10.  SUP_ALG_DEFAULT: the simultaneous
                              sweep, or the block-iterative one when block_iterative = 1 */
    int stop_enabled;      /* 1: the paper's default termination (A-25) is tested after
                              every sweep but the last: with P^k = Eq. 12 (p = 2) and f^k = f(x^k) at the iterate after sweep k-1,
                              stop iff (P^k <= prox_tol  or  |P^k - P^(k-1)| / max(1, P^(k-1)) < dprox_tol for n_consec
                              consecutive sweeps)  and, when an objective is perturbed,  |f^k - f^(k-1)| / max(1, f^(k-1)) < dobj_tol.
                              n_iter is the paper's N_max.  After a stop the remaining sweeps are skipped on the device (x stays
                              the iterate the rule was met at); sup_get_state reports n_done and stop_reason */
    double prox_tol;       /* paper's default 1e-6 */
    double dprox_tol;      /* paper's default 1e-8 */
    int n_consec;          /* paper's default 5 */
    double dobj_tol;       /* paper's default 1e-6 */
    int step_rule;         /* sup_step_rule: how beta_k is chosen.  SUP_RULE_POWER (0): beta0 * a^l with the accept test (Alg. 1) */
    double f_ref;          /* SUP_RULE_ADAPTIVE: Eq. 11's reference value at the start of the run (resume state: pass the f_ref
                              sup_get_state reported) */
    double f_ref_shrink;   /* SUP_RULE_ADAPTIVE: in (0, 1]; when a perturbation phase starts at f(x^k) <= f_ref the reference
                              becomes f_ref_shrink * f(x^k) after the phase (A-30) */
} sup_options;

/* feasibility-seeking operators (PAPER.md Table A.5) */
typedef enum {
    SUP_ALG_DEFAULT = 0, /* simultaneous projection x - lambda A^T D c(x) (A-1), or block-iterative (A-14) */
    SUP_ALG_DROP = 2,    /* x - lambda Z A^T M c(x), M = diag(w_i), Z = diag(1/nnz(A_:,j))  (L602, L608; A-26) */
    SUP_ALG_EMR = 3      /* x - (||p||^2 / ||M^(1/2) A p||^2) p,  p = A^T M c(x)             (L605; A-26); lambda is not used */
} sup_algorithm;

/* final state of a run, read back by sup_get_state (host struct) */
typedef struct {
    int64_t ell;         /* step-size exponent after the run */
    int64_t k;           /* number of sweeps done since k0 (absolute index of the next sweep) */
    int64_t n_trials;    /* trials since the last sup_superiorize / sup_perturb_* call started */
    int64_t n_decisions; /* entries written to `decisions` (may exceed the capacity: then only the first cap are stored) */
    int32_t warn;        /* bit 0: a reduction step hit J_max = 10000 trials and was skipped (A-12) */
    int32_t fault;       /* bit 0: device-side barrier timed out; bit 1: non-finite objective */
    double f;            /* objective value carried by the last perturbation phase */
    int64_t n_done;      /* sweeps actually performed by the last sup_superiorize call (< n_iter iff the stopping rule fired) */
    int32_t stop_reason; /* 0: ran all sweeps; else 1 * (P <= prox_tol) + 2 * (n_consec small changes) + 4 * (objective change small) */
    double step;         /* EMR: the last relaxation factor ||p||^2 / ||M^(1/2) A p||^2 */
    double f_ref;        /* SUP_RULE_ADAPTIVE: Eq. 11's reference value after the run */
} sup_state;

/* Bytes of workspace for `kind` on a matrix of the given shape (for SUP_WS_BLOCKS pass A's shape; for SUP_WS_DOSE
 * pass D_body's shape).  n_blocks is read for SUP_WS_BLOCKS only.  Both sizes are multiples of 256. */
sup_status sup_workspace_bytes(int kind, int64_t m, int64_t n, int64_t nnz, int dtype, int n_blocks,
                               size_t* persistent_bytes, size_t* scratch_bytes);

/* O-SETUP (A-3, A-4): normalises the weights (NULL => 1/m), computes ||a_i||^2 and
 * d_i = w_i/||a_i||^2 (0 for empty rows), validates the inputs, builds the explicit transposed CSR of A
 * (stable: every row of A^T is sorted by original row index).  Synchronises the stream. */
sup_status sup_create(sup_handle* out, const sup_csr* A, const void* lb, const void* ub, /* [m] */
                      const void* box_lo, const void* box_hi,                            /* [n] */
                      const void* weights,                                               /* [m] or NULL */
                      int dtype, void* workspace, size_t workspace_bytes, void* scratch, size_t scratch_bytes,
                      void* cuda_stream);

/* Block-iterative structure (PAPER.md:L54 BIP family; A-14): rows of A are block-contiguous, block t = rows
 * [block_rowptr[t], block_rowptr[t+1]).  Builds per-block transposed CSRs and the block-renormalised row scaling
 * (w_i / W_t) / ||a_i||^2.  block_rowptr is a HOST array [n_blocks+1].  Synchronises the stream. */
sup_status sup_set_blocks(sup_handle h, int n_blocks, const int64_t* block_rowptr, void* workspace,
                          size_t workspace_bytes, void* scratch, size_t scratch_bytes);

/* Dose objective matrix D_body (md x n CSR, same dtype; A-15): borrowed; builds its transposed CSR. */
sup_status sup_set_dose_matrix(sup_handle h, const sup_csr* D_body, void* workspace, size_t workspace_bytes,
                               void* scratch, size_t scratch_bytes);

/* How the dose objective's perturbation phase is evaluated.  mode 0 (default): through the Gram matrix G = D_body^T D_body when
 * sup_set_dose_matrix built it (it does when n <= 16384 and n^2 <= 2 nnz(D_body): f(x) = x^T G x, g = 2 G x, ||D g||^2 = g^T G g,
 * 1 + N dense n x n products per phase instead of 1 + 2N passes over D_body, K4d), else by matrix passes.
 * mode 1: always by matrix passes over D_body and its transpose.  Both are the same mathematics (A-15); they differ in rounding. */
sup_status sup_set_dose_mode(sup_handle h, int mode);

/* Which kernel runs the TV2D perturbation phase.  mode 0 (default): images of at least 8 rows and at most 4096 pixels per row block
 * of ny/8 rows (n <= 32768) take the CLUSTER kernel -- the image stays in the shared memory of 8 (or 16) CTAs for the whole phase, hardware
 * cluster barriers instead of a software grid barrier (K4s); larger images the cooperative grid kernel.
 * mode 1: always the grid kernel.  Same algorithm, same trial / decision / l sequence; sums in a different (fixed) order. */
sup_status sup_set_perturb_mode(sup_handle h, int mode);

/* Layout hint for the two gathered vectors (DESIGN.md section 4 "gather layouts").  The forward product gathers x and the
 * back-projection gathers y = D c(x) at the column / row indices of the nonzeros.  When an index space is a row-major
 * 2-D array -- x an image of x_shape = {rows, cols} pixels (rows * cols = n), the rows of A a sinogram of
 * y_shape = {angles, bins} (angles * bins = m) -- the library keeps its internal copies of x and y in 128-byte tiles of
 * 4 x 8 elements (fp64: 4 x 4) so that one warp's gathers along a ray touch few cache lines.  Either pointer may be NULL
 * (or {0, 0}): no hint for that side.  HOST arrays.  Pure data layout: every sum is formed from the same numbers in the
 * same order, results are bit-identical with and without the hint.  Rewrites the packed copies, drops the cached graph,
 * synchronises. */
sup_status sup_set_layout(sup_handle h, const int64_t* x_shape, const int64_t* y_shape);

/* Expert control of the two product kernels (S1+S2, S3), for tests and measurements: how many
 * lanes cooperate on one row of A (forward) and of A^T (backward).  -1: the planner's choice from the mean and the
 * longest row (default); 2, 4, 8, 16, 32: that many lanes of a warp per row (the planner's choice for rows of up to ~1000 entries:
 * 2 lanes up to ~60 entries per row, 32 from ~500); 64: a pair of warps per row; 128: CHUNKS -- a row is cut into pieces of 512 entries
 * that go to the warps round-robin, the last warp to finish a row adds the pieces in order (the planner's choice for rows of more
 * than 2048 entries on average, longest row <= 65536); 0: the whole CTA per row (rows longer than that); 1: SEGMENTS -- the warps
 * take fixed-size pieces of the matrix stream whatever rows they belong to (never chosen: slower, profiles/r02j_segments.md);
 * -2 (either argument): do not use the bulk-copy staged kernels at all but the plain group-per-row kernels.  A request that the longest row cannot satisfy is
 * widened by the planner.  Re-plans in place, drops the cached graph, synchronises the stream.  Results differ
 * between settings only by the summation order inside a row. */
sup_status sup_set_row_mode(sup_handle h, int lanes_forward, int lanes_backward);

/* n_sweeps simultaneous sweeps x <- P_box(x - lambda A^T D c(x)), in place (O-SWEEP; Eq. 2, 3; L427). */
sup_status sup_project_simultaneous(sup_handle h, void* x, double lambda, int n_sweeps);

/* The two halves of one simultaneous sweep as separate calls (what bench.py times one kernel at a time):
 * sup_forward_violation: S1+S2, y_i = d_i c_i(x) into the handle's internal y;  sup_backproject_update: S3,
 * x <- P_box(x - lambda A^T y) with that y.  Calling them in this order equals one sup_project_simultaneous sweep. */
sup_status sup_forward_violation(sup_handle h, const void* x);
sup_status sup_backproject_update(sup_handle h, void* x, double lambda);

/* The halves of a ROW-SHARDED sweep: every GPU owns a block of rows of A (its own handle, created on that
 * block) and a replica of x.  sup_forward_violation(h, x) forms the block's y; sup_backproject_partial writes the block's
 * share u = scale * A_block^T y (length n, plain order, not applied) -- scale = the block's share of the global weights, because
 * a handle normalises its weights over its own rows; the caller sums the u of all blocks (one all-reduce of an n-vector);
 * sup_apply_update then does x <- P_box(x - lambda u) identically on every GPU (Eq. 3). */
sup_status sup_backproject_partial(sup_handle h, void* u, double scale);
sup_status sup_apply_update(sup_handle h, void* x, const void* u, double lambda);

/* n_sweeps DROP sweeps (Table A.5): x <- P_box(x - lambda Z A^T M c(x)); for equality rows lb = ub = b the
 * residual c(x) is A x - b, the table's formula (A-26). */
sup_status sup_project_drop(sup_handle h, void* x, double lambda, int n_sweeps);

/* n_sweeps EMR sweeps (Table A.5): x <- P_box(x - t p), p = A^T M c(x), t = ||p||^2 / ||M^(1/2) A p||^2 --
 * three matrix passes per sweep (A, A^T, A) with the two norms reduced inside the product kernels.  Needs the staged kernels. */
sup_status sup_project_emr(sup_handle h, void* x, int n_sweeps);

/* n_sweeps block-iterative sweeps (O-BLOCK-SWEEP), in place. */
sup_status sup_block_iterative(sup_handle h, void* x, double lambda, int n_sweeps);

/* One perturbation phase (Alg. 1 lines 4-17) with the TV objective, step policy PER_TRIAL:
 * N accepted reduction steps from x, in place.  dims = 1 (shape[0] = n), 2 (shape = {ny, nx}) or 3 (shape = {nz, ny, nx}); shape is a HOST
 * array.  *ell (HOST) is read as the starting exponent and overwritten with the final one.  Synchronises. */
sup_status sup_perturb_tv(sup_handle h, void* x, int dims, const int64_t* shape, int N, double beta0, double a,
                          int64_t* ell);

/* Same with the dose objective ||D_body x||^2 (needs sup_set_dose_matrix). */
sup_status sup_perturb_dose(sup_handle h, void* x, int N, double beta0, double a, int64_t* ell);

/* Same with the mean objective f_Mean = (1/N_S) sum_{i in S} (D_S x)_i (Eq. 21), D_S being the matrix given
 * to sup_set_dose_matrix.  The objective is linear, its gradient (1/N_S) D_S^T 1 is formed once at sup_set_dose_matrix, and
 * every first trial is accepted: the phase is N axpy steps. */
sup_status sup_perturb_mean(sup_handle h, void* x, int N, double beta0, double a, int64_t* ell);

/* One perturbation phase with Eq. 11's step size (SUP_RULE_ADAPTIVE above): N steps
 * x <- x - ((f(x) - f_ref)/||g||^2) g, each only while f(x) > *f_ref and g != 0.  objective: SUP_OBJ_TV1D / TV2D / TV3D (shape as
 * in sup_options) or SUP_OBJ_DOSE.  *f_ref (HOST) is read and, by the rule of DESIGN.md A-30, updated.  x in place.
 * Synchronises.  SUP_ERR_INVALID_ARG for other objectives, shrink outside (0, 1] or a non-finite *f_ref. */
sup_status sup_perturb_adaptive(sup_handle h, void* x, int objective, const int64_t* shape, int N, double* f_ref, double shrink);

/* Algorithm 1, Eq. 10 (L91): for k = k0 .. k0+n_iter-1: perturbation phase of N reduction steps
 * (beta = beta0 * a^l), then one sweep.  x in place.  N = 0 or objective NONE gives the basic algorithm.
 * Asynchronous; read the final state with sup_get_state. */
sup_status sup_superiorize(sup_handle h, void* x, int n_iter, int N, double beta0, double a, const sup_options* opt);

/* Same run with x in HOST memory (pinned for best speed): copies x to the device, runs, copies it back and
 * synchronises.  This is the end-to-end entry bench.py times as "e2e". */
sup_status sup_superiorize_host(sup_handle h, void* x_host, int n_iter, int N, double beta0, double a,
                                const sup_options* opt);

/* Synchronises and copies the device-side run state to *out (HOST). */
sup_status sup_get_state(sup_handle h, sup_state* out);

/* Proximity of x (O-PROX): mode 0 = 1/2 sum w_i dist_i^2 (Eq. 5), mode 1 = sum w_i dist_i^p (L211 Eq. 12),
 * mode 2 = max_i dist_i (L215 Eq. 13); dist_i = |c_i| / ||a_i|| (0 for empty rows).  *out is HOST.  Synchronises. */
sup_status sup_proximity(sup_handle h, const void* x, int mode, double p, double* out);

/* Objective value f(x) for `kind` (sup_objective_kind); shape is a HOST array (TV2D: {ny, nx}).  *out is HOST. */
sup_status sup_objective(sup_handle h, const void* x, int kind, const int64_t* shape, double* out);

/* The ONE entry point that allocates nothing and needs no handle: the TV2D objective value f(X) of PAPER.md:L308-311 Eq. 15
 * (= sup_objective(h, x, SUP_OBJ_TV2D, {ny, nx}, .)), for callers that cannot call cudaMalloc at that point (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  Its scratch -- one partial sum per image row and an arrival counter --
 * is a file-scope __device__ array of SUP_STATIC_MAX_ROWS doubles (128 KB) that every GPU which loads the library holds until the
 * process exits; no cudaMalloc, cudaFree or allocating library routine is called.
 *   x        DEVICE, [ny*nx] row-major, of type `dtype` (SUP_F32 / SUP_F64), on the CURRENT device (checked);
 *   out_dev  DEVICE, one double, written by the kernel;   stream: cudaStream_t as void* (NULL = default stream).
 * Asynchronous (the value is in *out_dev when the stream reaches that point).  ny > SUP_STATIC_MAX_ROWS or nx > 2^31 is refused with
 * SUP_ERR_INVALID_ARG before any launch (text through sup_last_error(NULL)).  Terms and sums in fp64, fixed summation order (row
 * sums, then the rows in order): the value differs from sup_objective's by the summation order only.
 * The scratch is SHARED by all calls on a device and keeps the last call's contents; each call clears the counter and overwrites
 * every row slot it reads.  Calls that OVERLAP on one GPU (different streams or host threads) RACE on it: serialise them. */
#define SUP_STATIC_MAX_ROWS 16384
sup_status sup_tv2d_value_static(const void* x, int dtype, int64_t ny, int64_t nx, double* out_dev, void* stream);

/* Copies derived arrays for inspection/tests: which = 0: d [m] (dtype); 1: A^T rowptr [n+1] int64;
 * 2: A^T col [nnz] int32 (original row indices); 3: A^T val [nnz] (dtype); 5: y [m] (dtype), the scaled violation
 * d_i c_i(x) left by the last forward product (sup_forward_violation or a sweep).  dst is a DEVICE pointer. */
sup_status sup_get_derived(sup_handle h, int which, void* dst, size_t dst_bytes);

/* Number of kernel launches this handle has enqueued so far (graph replays count their kernel nodes). */
int64_t sup_launch_count(sup_handle h);

const char* sup_last_error(sup_handle h);
sup_status sup_destroy(sup_handle h);
const char* sup_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SUP_H */
