// sup_internal.cuh -- shared declarations of libsup's translation units (not part of the public ABI).
// Method and readings: include/sup.h, DESIGN.md.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <set>
#include <vector>

#include "sup.h"

#define SUP_THREADS 256          // threads per CTA of every kernel
#define SUP_MAX_PARTIALS 2048    // upper bound on the grid of any kernel that feeds a two-stage reduction
#define SUP_J_MAX 10000          // trials per reduction step (A-12)

// Plan of the bulk-copy-staged SpMV (sup_stream.cu) for one row range of one matrix: persistent CTA b owns rows
// [part[b], part[b+1]) -- contiguous, balanced by nonzeros.  ok = false: the range does not qualify (a row too
// long for the ring, misaligned arrays) and the group-per-row kernels of sup_spmv.cu are used instead.
#define SUP_STREAM_NBMAX 4096  // upper bound on the persistent grid
struct StreamPlan {
    const int64_t* part = nullptr;  // device, [nb + 1]
    int nb = 0;
    int G = 32;        // lanes per row
    bool ok = false;
    int64_t max_row = 0;
    void* table = nullptr;  // the persistent memory `part` lives in (kept so that sup_set_row_mode can re-plan in place)
};

struct CsrD {  // device CSR (borrowed or living in workspace)
    int64_t rows = 0, cols = 0, nnz = 0;
    const int64_t* rowptr = nullptr;
    const int32_t* col = nullptr;
    const void* val = nullptr;
    const void* pk = nullptr;  // fp32 handles: packed (value bits, column) pairs, 8 B per nonzero (sup_stream.cu); else NULL
    int64_t alloc_nnz = 0;  // length of the col/val arrays (>= nnz; per-block transposes share one pair of arrays)
    StreamPlan plan;  // plan for all rows
};

// device-resident run state; one per handle
struct DevState {
    long long ell;        // step-size exponent l
    long long k;          // absolute sweep index
    long long it;         // sweep index inside the current sup_superiorize run (row of `trace`)
    long long n_trials;   // trials since the run started
    long long sweep_trials;
    long long n_dec;      // decisions logged (may exceed cap)
    int warn;
    int fault;
    double f;             // objective carried by the last perturbation phase
    double apow;          // a^l as the running fp64 product (PER_TRIAL; A-20)
    double scalar_out;    // result slot of finalize kernels (proximity / objective)
    // the paper's stopping rule (A-25) and what the feasibility-seeking kernels leave for the next kernel
    double prox_prev, f_prev;  // P^(k-1), f^(k-1)
    double prox_cur, f_cur;    // P^k, f^k of the sweep being closed
    double step;          // EMR: ||p||^2 / ||M^(1/2) A p||^2 of the current sweep
    double cf;            // dose perturbation: coefficient of the accepted step (0: none)
    long long n_done;     // sweeps performed by this run
    long long n_iter;     // sweeps asked of this run (the rule is not applied after the last one)
    int consec;           // consecutive sweeps with a small relative proximity change
    int stop;             // 1: the rule fired -- every later kernel of the run returns at once
    int stop_reason;
    double f_ref;         // Eq. 11's reference value (adaptive step rule, A-30)
    double f_start;       // dose objective, adaptive rule: f at the start of the phase (decides the update of f_ref)
    // grid barrier of the perturbation kernel (grid_reduce, sup_perturb.cu), each field in a 128-byte line of its own
    alignas(128) unsigned long long bar_count;  // arrivals, monotone within a run
    alignas(128) unsigned long long bar_base;   // value of bar_count when the last launch's barriers were complete
};

// kernels that precede a product kernel in a sweep let it start early (sup_stream.cu: programmatic dependent launch)
__device__ __forceinline__ void sup_pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

struct Bump {  // bump allocator over caller-provided workspace
    char* base = nullptr;
    size_t cap = 0, off = 0;
    bool ok = true;
    void* take(size_t bytes) {
        size_t a = (bytes + 255) & ~size_t(255);
        if (off + a > cap) { ok = false; return nullptr; }
        void* p = base + off;
        off += a;
        return p;
    }
};

// Index swizzle of the forward gathers.  With a power-of-two image pitch (512 floats = 2 KB) the x entries a
// near-vertical ray gathers all have the same address modulo 128 B, i.e. sit in the same L1 data bank: measured, the
// chunks of the forward product at those angles run 1.6x slower than the median at pitch 512, 1.2x at 528, 1.08x at 520
// (profiles/r01c_staged.md).  XOR-ing the five bank bits of the index with a fold of the upper bits is a bijection
// inside every 128-byte line (sector membership is preserved too), and puts vertically adjacent pixels in different banks.
__host__ __device__ static inline int sup_swz(int j) { return j ^ (((j >> 9) ^ (j >> 14)) & 31); }

// Gather map: where element j of a gathered vector (the forward product's x, the back-projection's y) lives in the
// copy the kernels gather from.  A bijection of [0, size) chosen so that the gathers of one warp touch few 128-byte
// lines and distinct L1 data banks (profiles/r02c_layout.md):
//   kind 0  identity
//   kind 1  bank swizzle only (sup_swz): elements permuted inside each line
//   kind 2  the vector is a row-major R x C array (an image, a sinogram: sup_set_layout) stored as line-sized tiles of
//           th x tw elements (th * tw * element size = 128 B, tw elements = one 32-byte sector), so that a ray crossing
//           the image at any angle -- or a pixel's trace through the sinogram -- stays inside a tile for several
//           elements; inside a tile the position is XOR-ed with (tile row mod tw) | (tile column mod th) * tw, a
//           bijection that keeps sectors whole and puts vertically / horizontally adjacent tiles in different banks.
//           The R mod th last rows and C mod tw last columns do not fill whole tiles and follow the tiled region in
//           row-major order (no padding: the map stays onto [0, R*C)).
struct GMap {
    int kind = 0;
    int C = 1;          // columns of the 2-D view
    int Rm = 0, Cm = 0; // extent of the tiled region (multiples of th, tw)
    int ntc = 0;        // tiles per tile row = Cm / tw
    int th = 4, tw = 8; // powers of two (a 32-byte sector wide, four sectors high)
    int th_shift = 2, tw_shift = 3;
    unsigned long long Cmagic = 0;  // ceil(2^64 / C): j / C = mulhi64(j, Cmagic) exactly for every 32-bit j (device code; the
                                    // epilogue of every row of the product kernels maps an index: three runtime divisions there
                                    // were ~60 of the ~200 instructions a warp spends per row group outside the dot product)
};
__host__ __device__ static inline int sup_gmap(const GMap& M, int j) {
    if (M.kind == 0) return j;
    if (M.kind == 1) return sup_swz(j);
#ifdef __CUDA_ARCH__
    const int r = M.Cmagic ? int(__umul64hi((unsigned long long)(unsigned)j, M.Cmagic)) : j;  // (Cmagic = 0: C = 1)
#else
    const int r = j / M.C;
#endif
    const int c = j - r * M.C;
    const int main_count = M.Rm * M.Cm;
    if (r < M.Rm) {
        if (c < M.Cm) {
            const int tr = r >> M.th_shift, tc = c >> M.tw_shift;
            const int in = ((r & (M.th - 1)) << M.tw_shift) + (c & (M.tw - 1));
            const int v = (tr & (M.tw - 1)) | ((tc & (M.th - 1)) * M.tw);
            return (tr * M.ntc + tc) * (M.th * M.tw) + (in ^ v);
        }
        return main_count + r * (M.C - M.Cm) + (c - M.Cm);
    }
    return main_count + M.Rm * (M.C - M.Cm) + (r - M.Rm) * M.C + c;
}

struct sup_ctx {
    int dt = 0;
    size_t esz = 4;
    cudaStream_t stream = nullptr;
    int num_sms = 148;
    int64_t m = 0, n = 0, nnz = 0;
    CsrD A, AT;
    const void *lb = nullptr, *ub = nullptr, *lo = nullptr, *hi = nullptr;
    void* d = nullptr;          // [m] dtype: w_i / ||a_i||^2
    double* w = nullptr;        // [m] normalised weights
    double* invnorm = nullptr;  // [m] 1/||a_i|| (0 for empty rows)
    void* y = nullptr;          // [m] dtype: scaled violation d_i c_i
    void* g = nullptr;          // [n] dtype: gradient of the objective
    void* x2 = nullptr;         // [n] dtype: second iterate buffer of the perturbation kernel (deferred accepted steps)
    void* g2 = nullptr;         // [n] dtype: second gradient buffer
    void* xdev = nullptr;       // [n] dtype: staging copy of x for sup_superiorize_host
    double* partials = nullptr; // [2][SUP_MAX_PARTIALS]
    DevState* state = nullptr;
    int g_fwd = 32, g_bwd = 32; // lanes per row of the two products
    // De-aliased mirror of x for the forward gathers (sup_stream.cu): xg[sup_swz(j)] = x[j], colg = sup_swz(A.col).
    int32_t* colg = nullptr;    // [nnz]  (fp64 handles; fp32 handles carry the swizzled column inside A.pk)
    void* pk_a = nullptr;       // [nnz] x 8 B, fp32 handles: (val, sup_swz(col)) of A
    void* pk_at = nullptr;      // [nnz] x 8 B, fp32 handles: (val, row) of A^T
    void* pk_atb = nullptr;     // [nnz] x 8 B, fp32 handles: the per-block transposes (sup_set_blocks)
    void* pk_d = nullptr;       // [nnz_D] x 8 B, fp32 handles: D_body and its transpose (sup_set_dose_matrix), plain indices
    void* pk_dt = nullptr;
    void* wT = nullptr;         // [m] dtype: the normalised weights w_i (M of DROP / EMR)
    void* zcol = nullptr;       // [n] dtype: 1 / nnz(A_:,j), 0 for an empty column (Z of DROP)
    const int* stop_ptr = nullptr;  // &state->stop while a run with the stopping rule is being enqueued, else NULL
    double* red = nullptr;      // [3][SUP_STREAM_NBMAX] per-CTA partials of the product kernels' reductions
    void* xg = nullptr;         // [n rounded up to 512] dtype: xg[sup_gmap(xmap, j)] = x[j]
    GMap xmap, ymap;            // maps in force: x mirror read by the staged forward product; internal y (identity unless every
                                // product runs on the staged fp32 kernels, which read y through the packed A^T)
    GMap ymap_req;              // what sup_set_layout asked for on the row side
    bool xg_synced = false;     // enqueue-time flag: xg mirrors x (set by the back-projection, cleared when x changes elsewhere)
    int stream_nb = 0;          // persistent grid of the row-stream kernels (-1: unavailable)
    bool use_stream = true;     // false: the group-per-row kernels of sup_spmv.cu (sup_set_row_mode(h, -2, -2))
    int lanes_fwd = -1, lanes_bwd = -1;      // sup_set_row_mode overrides of the lanes per row (-1: planner's choice)
    std::set<const void*> smem_opted_in;     // kernels already opted in to > 48 KB dynamic shared memory on this handle's device
    int device = 0;             // CUDA device of the workspace; every entry point runs with it current
    // block-iterative
    int n_blocks = 0;
    std::vector<int64_t> block_rowptr;
    std::vector<CsrD> ATb;
    std::vector<int> g_bwd_blk;
    std::vector<StreamPlan> stream_fwd_blk;  // forward product restricted to block t's rows of A
    void* d_blk = nullptr;      // [m] dtype: (w_i/W_t)/||a_i||^2
    // dose objective
    bool has_dose = false;
    CsrD D, DT;
    void* r_dose = nullptr;     // [md] dtype
    void* q_dose = nullptr;     // [md] dtype: D g
    void* gmean = nullptr;      // [n] dtype: (1/N_S) D_S^T 1, the constant gradient of f_Mean (Eq. 21)
    double* gmean_norm2 = nullptr;  // device scalar ||gmean||^2
    void* gram = nullptr;           // [n][gram_ld] G = D^T D of the dose matrix (sup_gram.cu), NULL when not applicable
    int64_t gram_ld = 0;
    void* gram_w = nullptr;         // [n] G g of the current reduction step
#ifdef SUP_NO_PDL
    bool pdl = false;
#else
    bool pdl = true;                // programmatic dependent launch between consecutive k_staged launches (sup_stream.cu)
#endif
    int cluster16 = 0;              // thread-block clusters of 16 for the small-image perturbation kernel: 0 not asked yet, 1 yes, -1 no
    int perturb_mode = 0;           // 0: small TV2D images take the cluster kernel (sup_perturb_small.cu), 1: always the grid kernel
    int dose_mode = 0;              // 0: Gram path when available, 1: matrix passes over D and D^T (sup_set_dose_mode)
    int g_d = 8, g_dt = 32;
    // cached graph of one superiorized sweep
    cudaGraphExec_t gexec = nullptr;
    cudaGraph_t graph = nullptr;
    int graph_nodes = 0;
    bool graph_failed = false;
    struct GraphKey {
        const void* x = nullptr;
        int N = 0, objective = 0, block = 0, policy = 0, trace_mode = 0;
        int64_t n_restart = 0;
        int algorithm = 0, stop = 0, n_consec = 0, step_rule = 0;
        double tols[3] = {0, 0, 0}, shrink = 0;
        double beta0 = 0, a = 0, lambda = 0;
        int64_t s0 = 0, s1 = 0, s2 = 0;
        const void *trace = nullptr, *dec = nullptr, *decf = nullptr;
        int64_t cap = 0;
        bool operator==(const GraphKey& o) const {
            return x == o.x && N == o.N && objective == o.objective && block == o.block && policy == o.policy &&
                   trace_mode == o.trace_mode && beta0 == o.beta0 && a == o.a && lambda == o.lambda && s0 == o.s0 &&
                   s1 == o.s1 && s2 == o.s2 && algorithm == o.algorithm && stop == o.stop && n_consec == o.n_consec &&
                   tols[0] == o.tols[0] && tols[1] == o.tols[1] && tols[2] == o.tols[2] && trace == o.trace && dec == o.dec && decf == o.decf && cap == o.cap && n_restart == o.n_restart &&
                   step_rule == o.step_rule && shrink == o.shrink;
        }
    } gkey;
    int64_t launches = 0;
    char err[512] = {0};
};

sup_status sup_fail(sup_ctx* h, sup_status s, const char* fmt, ...);
extern char g_create_error[512];

#define SUP_CUDA(h, call)                                                                            \
    do {                                                                                             \
        cudaError_t e__ = (call);                                                                    \
        if (e__ != cudaSuccess)                                                                      \
            return sup_fail((h), SUP_ERR_CUDA, "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e__)); \
    } while (0)

static inline int sup_pick_group(int64_t nnz, int64_t rows) {
    // lanes cooperating on one row: about a quarter of the mean row length, a power of two in [4, 32]
    double avg = rows > 0 ? double(nnz) / double(rows) : 0.0;
    int g = 4;
    while (g < 32 && avg > 4.0 * g) g <<= 1;
    return g;
}
static inline int sup_grid_for(int64_t work_items, int per_block, int cap) {
    int64_t b = (work_items + per_block - 1) / per_block;
    if (b < 1) b = 1;
    if (b > cap) b = cap;
    return int(b);
}

// ---- setup (sup_setup.cu) ---------------------------------------------------------------------------------
size_t sup_transpose_scratch_bytes(int64_t nnz, int64_t cols, size_t esz);
// transposes rows [r0, r1) of A into `out` (cols x (r1-r0) CSR whose "col" entries are ORIGINAL row indices);
// out arrays must be preallocated: rowptr [A.cols+1], col/val [nnz of the row range].  Stable in row order.
sup_status sup_transpose_rows(sup_ctx* h, const CsrD& A, int64_t r0, int64_t r1, int64_t e0, int64_t e1,
                              int64_t* out_rowptr, int32_t* out_col, void* out_val, int64_t out_base, void* scratch,
                              size_t scratch_bytes);
sup_status sup_setup_rows(sup_ctx* h, const void* weights, void* scratch, size_t scratch_bytes);
sup_status sup_setup_block_scaling(sup_ctx* h, void* scratch, size_t scratch_bytes);
sup_status sup_validate(sup_ctx* h, const CsrD& A, bool check_bounds, void* scratch);

// ---- products (sup_spmv.cu) -------------------------------------------------------------------------------
// red_out (forward): per-CTA partials of sum c_i y_i, only produced by the staged kernel (NULL otherwise)
void sup_launch_fwd(sup_ctx* h, const void* x, int64_t r0, int64_t r1, const void* dscale, const StreamPlan* rp, double* red_out = nullptr);
void sup_launch_bwd(sup_ctx* h, const CsrD& AT, int G, void* x, double lambda, const void* zscale = nullptr);
void sup_launch_proximity(sup_ctx* h, const void* x, int mode, double p, double* out_dev);

// ---- bulk-copy-staged products (sup_stream.cu) ---------------------------------------------------------------
size_t sup_stream_table_bytes();  // bytes of one partition table (256-aligned)
// Plans rows [r0, r1) of M: grid size, partition table (written into `table`, sup_stream_table_bytes() bytes of
// persistent workspace), lanes per row; `forward` only selects which tuning overrides apply; synchronises the stream.  `scratch` needs 256 bytes.
sup_status sup_stream_plan(sup_ctx* h, const CsrD& M, int64_t r0, int64_t r1, bool forward, void* table, void* scratch,
                           StreamPlan* out);
void sup_launch_staged(sup_ctx* h, int mode, const StreamPlan& sp, const CsrD& M, const void* vec, const void* p1, const void* p2,
                       const void* p3, void* out, void* out2, double lambda, const GMap& omap, bool deep, double* red_out);
void sup_launch_stream_fwd(sup_ctx* h, const StreamPlan& rp, const void* x, const void* dscale, double* red_out);
void sup_launch_stream_bwd(sup_ctx* h, const CsrD& AT, const StreamPlan& rp, void* x, double lambda, const void* zscale);
void sup_launch_stream_plain_A(sup_ctx* h, const void* v_g, void* out, double scale, const void* wrow, double* red_out);
void sup_launch_stream_plain_AT(sup_ctx* h, void* out_g, double scale, double* red_out);
sup_status sup_stream_setup_gather(sup_ctx* h);  // fills colg (fp64) or the packed copy of A (fp32) from A.col / A.val through xmap
// fp32 handles: dst[k] = (val[k], sup_gmap(map, col[k])) for k in [0, nnz)
sup_status sup_stream_pack(sup_ctx* h, const void* val, const int32_t* col, int64_t nnz, void* dst, const GMap& map);
// (re)decides ymap and (re)writes every packed / mapped copy the staged kernels read; call after plans or maps change
sup_status sup_stream_refresh_layout(sup_ctx* h);
void sup_launch_unmap(sup_ctx* h, const void* src, void* dst, int64_t count, const GMap& map);  // dst[i] = src[map(i)]
bool sup_stream_forward_uses_xg(const sup_ctx* h);

// ---- perturbation (sup_perturb.cu) ------------------------------------------------------------------------
struct PerturbParams {
    int objective;
    int64_t nz, ny, nx;
    int N;
    double beta0, a;
    int policy;
    int8_t* decisions;
    double* decision_f;
    int64_t cap;
    int64_t n_restart;
    bool write_mirror;  // also write the final iterate to the gather mirror of x (xg_synced stays true)
    int step_rule = 0;  // sup_step_rule
    double shrink = 1.0;
};
sup_status sup_launch_perturb(sup_ctx* h, void* x, const PerturbParams& pp);
void sup_launch_objective(sup_ctx* h, const void* x, int kind, int64_t nz, int64_t ny, int64_t nx, double* out_dev);
void sup_launch_begin_run(sup_ctx* h, int64_t ell0, int64_t k0, double a, int64_t n_iter = 0, double f_ref = 0.0);
int sup_perturb_grid(sup_ctx* h, int objective);
bool sup_perturb_small_eligible(const sup_ctx* h, const PerturbParams& pp);
sup_status sup_launch_perturb_small(sup_ctx* h, void* x, const PerturbParams& pp);

// ---- DROP / EMR, stopping rule, f_Mean (sup_algos.cu) ---------------------------------------------------------------
sup_status sup_setup_wz(sup_ctx* h);
void sup_launch_emr_update(sup_ctx* h, const double* red_pp, int np_pp, const double* red_qq, int np_qq, const void* p_g, void* x);
// mode: 0 after a sweep with (P, f) measured, 1 run start, 2 before the back-projection (basic algorithm), 3 after a sweep with
// nothing measured, 4 after the run (see k_close_sweep); np = 0: P from st->prox_cur
void sup_launch_close_sweep(sup_ctx* h, double* trace, const double* red_prox, int np, int mode, int use_f, int perturbed,
                            const sup_options& o);
sup_status sup_setup_mean_gradient(sup_ctx* h);
sup_status sup_launch_perturb_mean(sup_ctx* h, void* x, const PerturbParams& pp);
int sup_launch_mean_value(sup_ctx* h, const void* x);
sup_status sup_launch_perturb_dose_staged(sup_ctx* h, void* x, const PerturbParams& pp);

// ---- dose objective through the Gram matrix (sup_gram.cu) -------------------------------------------------------------------------
bool sup_gram_applicable(int64_t n, int64_t nnz);
int64_t sup_gram_ld(int64_t n);
sup_status sup_gram_build(sup_ctx* h);
sup_status sup_launch_perturb_dose_gram(sup_ctx* h, void* x, const PerturbParams& pp);
