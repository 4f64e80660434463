// sup_api.cu -- the C ABI of libsup (include/sup.h): argument checks, workspace layout, the sweep loops
// (O-SWEEP, O-BLOCK-SWEEP, O-SUPERIORIZE of DESIGN.md) and CUDA-graph capture of one superiorized sweep (S8).
#include <cmath>
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "sup_internal.cuh"

static size_t al(size_t b) { return (b + 255) & ~size_t(255); }

extern "C" const char* sup_version(void) { return "libsup 0.1 (sm_100a)"; }

extern "C" const char* sup_last_error(sup_handle h) { return h ? h->err : g_create_error; }

extern "C" int64_t sup_launch_count(sup_handle h) { return h ? h->launches : 0; }

extern "C" sup_status sup_workspace_bytes(int kind, int64_t m, int64_t n, int64_t nnz, int dtype, int n_blocks,
                                          size_t* persistent_bytes, size_t* scratch_bytes) {
    if (m <= 0 || n <= 0 || nnz < 0 || (dtype != SUP_F32 && dtype != SUP_F64) || !persistent_bytes || !scratch_bytes)
        return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_workspace_bytes: bad argument");
    const size_t esz = dtype == SUP_F32 ? 4 : 8;
    size_t p = 0, s = 0;
    switch (kind) {
        case SUP_WS_CREATE:
            p = al(size_t(n + 1) * 8) + al(size_t(nnz) * 4) + al(size_t(nnz) * esz)  // A^T
                + al(size_t(m) * esz)                                                // d
                + 2 * al(size_t(m) * 8)                                              // w, 1/||a||
                + al(size_t(m) * esz) + 4 * al(size_t(n) * esz)                      // y, g, xdev, x2, g2
                + al(2 * SUP_MAX_PARTIALS * 8) + al(sizeof(DevState)) + 2 * sup_stream_table_bytes()
                + (dtype == SUP_F32 ? 2 * al(size_t(nnz) * 8) : al(size_t(nnz) * 4))               // packed A, A^T (fp32) | colg (fp64)
                + al(size_t((n + 511) & ~int64_t(511)) * esz)                                      // xg
                + al(size_t(m) * esz) + al(size_t(n) * esz)                                        // wT, zcol (DROP / EMR)
                + al(3 * size_t(SUP_STREAM_NBMAX) * 8)                                             // reduction partials of the product kernels
                + 1024;
            s = sup_transpose_scratch_bytes(nnz, n, esz) + 4096;
            break;
        case SUP_WS_BLOCKS:
            if (n_blocks < 1) return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_workspace_bytes: n_blocks < 1");
            p = size_t(n_blocks) * al(size_t(n + 1) * 8) + al(size_t(nnz) * 4) + al(size_t(nnz) * esz) + al(size_t(m) * esz) +
                2 * size_t(n_blocks) * sup_stream_table_bytes() + (dtype == SUP_F32 ? al(size_t(nnz) * 8) : 0) + 1024;
            s = sup_transpose_scratch_bytes(nnz, n, esz) + al(size_t(n_blocks) * 8) + 4096;
            break;
        case SUP_WS_DOSE:  // (m, n, nnz) describe D_body
            p = al(size_t(n + 1) * 8) + al(size_t(nnz) * 4) + al(size_t(nnz) * esz) + 2 * al(size_t(m) * esz)
                + al(size_t(n) * esz) + 256                                                        // gradient of f_Mean and its norm
                + (dtype == SUP_F32 ? 2 * al(size_t(nnz) * 8) : 0) + 2 * sup_stream_table_bytes()  // packed D, D^T; partition tables
                + (sup_gram_applicable(n, nnz) ? al(size_t(n) * size_t(sup_gram_ld(n)) * esz) + al(size_t(n) * esz) : 0)  // G = D^T D, G g
                + 1024;
            s = sup_transpose_scratch_bytes(nnz, n, esz) + 4096;
            break;
        default:
            return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_workspace_bytes: unknown kind");
    }
    *persistent_bytes = al(p);
    *scratch_bytes = al(s);
    return SUP_OK;
}

static bool aligned256(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 255u) == 0; }

// Every entry point runs with the handle's device current (the device the workspace lives on) and restores the caller's.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};
#define SUP_ENTER(h) DeviceGuard guard__((h)->device)

extern "C" sup_status sup_create(sup_handle* out, const sup_csr* A, const void* lb, const void* ub, const void* box_lo,
                                 const void* box_hi, const void* weights, int dtype, void* workspace, size_t workspace_bytes,
                                 void* scratch, size_t scratch_bytes, void* cuda_stream) {
    if (!out) return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_create: out is NULL");
    *out = nullptr;
    if (!A || !A->rowptr || !A->col || !A->val || !lb || !ub || !box_lo || !box_hi)
        return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_create: NULL array argument");
    // rows and columns are 32-bit indices; the number of stored entries may exceed 2^31 (row pointers are 64-bit; the transpose
    // ranks entries with 32-bit unsigned positions, hence the 2^32 - 1 limit)
    if (A->m <= 0 || A->n <= 0 || A->nnz < 0 || A->n > 0x7fffffffLL || A->m > 0x7fffffffLL || A->nnz > 0xfffffffeLL)
        return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_create: m, n must be in [1, 2^31), nnz in [0, 2^32 - 1)");
    if (dtype != SUP_F32 && dtype != SUP_F64) return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_create: bad dtype");
    size_t need_p = 0, need_s = 0;
    sup_workspace_bytes(SUP_WS_CREATE, A->m, A->n, A->nnz, dtype, 1, &need_p, &need_s);
    if (!workspace || !scratch || workspace_bytes < need_p || scratch_bytes < need_s || !aligned256(workspace) || !aligned256(scratch))
        return sup_fail(nullptr, SUP_ERR_WORKSPACE, "sup_create: workspace needs %zu + %zu scratch bytes, 256-byte aligned", need_p, need_s);
    int dev = 0;
    cudaDeviceProp prop;
    cudaPointerAttributes pattr;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return sup_fail(nullptr, SUP_ERR_CUDA, "sup_create: no usable CUDA device (libsup has no CPU fallback)");
    }
    // the handle lives on the device that owns the workspace, whatever device is current in the calling thread
    if (cudaPointerGetAttributes(&pattr, workspace) == cudaSuccess && pattr.type == cudaMemoryTypeDevice) dev = pattr.device;
    else cudaGetLastError();
    DeviceGuard guard(dev);
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return sup_fail(nullptr, SUP_ERR_CUDA, "sup_create: cannot query device %d", dev);
    }
    sup_ctx* h = new (std::nothrow) sup_ctx;
    if (!h) return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_create: out of host memory");
    h->device = dev;
    h->dt = dtype;
    h->esz = dtype == SUP_F32 ? 4 : 8;
    h->stream = static_cast<cudaStream_t>(cuda_stream);
    h->num_sms = prop.multiProcessorCount;
    h->m = A->m;
    h->n = A->n;
    h->nnz = A->nnz;
    h->A.rows = A->m;
    h->A.cols = A->n;
    h->A.nnz = A->nnz;
    h->A.rowptr = A->rowptr;
    h->A.col = A->col;
    h->A.val = A->val;
    h->lb = lb;
    h->ub = ub;
    h->lo = box_lo;
    h->hi = box_hi;
    h->g_fwd = sup_pick_group(h->nnz, h->m);
    h->g_bwd = sup_pick_group(h->nnz, h->n);

    Bump B{static_cast<char*>(workspace), workspace_bytes, 0, true};
    int64_t* at_rowptr = static_cast<int64_t*>(B.take(size_t(h->n + 1) * 8));
    int32_t* at_col = static_cast<int32_t*>(B.take(size_t(h->nnz) * 4));
    void* at_val = B.take(size_t(h->nnz) * h->esz);
    h->d = B.take(size_t(h->m) * h->esz);
    h->w = static_cast<double*>(B.take(size_t(h->m) * 8));
    h->invnorm = static_cast<double*>(B.take(size_t(h->m) * 8));
    h->y = B.take(size_t(h->m) * h->esz);
    h->g = B.take(size_t(h->n) * h->esz);
    h->xdev = B.take(size_t(h->n) * h->esz);
    h->x2 = B.take(size_t(h->n) * h->esz);
    h->g2 = B.take(size_t(h->n) * h->esz);
    h->partials = static_cast<double*>(B.take(2 * SUP_MAX_PARTIALS * 8));
    h->state = static_cast<DevState*>(B.take(sizeof(DevState)));
    void* tab_a = B.take(sup_stream_table_bytes());
    void* tab_at = B.take(sup_stream_table_bytes());
    if (dtype == SUP_F32) {
        h->pk_a = B.take(size_t(h->nnz) * 8);
        h->pk_at = B.take(size_t(h->nnz) * 8);
    } else {
        h->colg = static_cast<int32_t*>(B.take(size_t(h->nnz) * 4));
    }
    h->xg = B.take(size_t((h->n + 511) & ~int64_t(511)) * h->esz);
    h->wT = B.take(size_t(h->m) * h->esz);
    h->zcol = B.take(size_t(h->n) * h->esz);
    h->red = static_cast<double*>(B.take(3 * size_t(SUP_STREAM_NBMAX) * 8));
    h->A.alloc_nnz = h->nnz;
    sup_status rc = SUP_OK;
    if (!B.ok) rc = sup_fail(h, SUP_ERR_WORKSPACE, "sup_create: workspace too small");
    if (rc == SUP_OK && cudaMemsetAsync(h->state, 0, sizeof(DevState), h->stream) != cudaSuccess)
        rc = sup_fail(h, SUP_ERR_CUDA, "sup_create: cannot touch the workspace: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc == SUP_OK) rc = sup_setup_rows(h, weights, scratch, scratch_bytes);
    if (rc == SUP_OK)
        rc = sup_transpose_rows(h, h->A, 0, h->m, 0, h->nnz, at_rowptr, at_col, at_val, 0, scratch, scratch_bytes);
    if (rc == SUP_OK && cudaStreamSynchronize(h->stream) != cudaSuccess)
        rc = sup_fail(h, SUP_ERR_CUDA, "sup_create: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc != SUP_OK) {
        memcpy(g_create_error, h->err, sizeof(g_create_error));
        delete h;
        return rc;
    }
    h->AT.rows = h->n;
    h->AT.cols = h->m;
    h->AT.nnz = h->nnz;
    h->AT.rowptr = at_rowptr;
    h->AT.col = at_col;
    h->AT.val = at_val;
    h->AT.alloc_nnz = h->nnz;
    h->A.pk = h->pk_a;
    h->AT.pk = h->pk_at;
    h->xmap.kind = 1;  // bank swizzle only, until sup_set_layout says what the index spaces look like
    rc = sup_stream_plan(h, h->A, 0, h->m, true, tab_a, scratch, &h->A.plan);
    if (rc == SUP_OK && cudaMemsetAsync(h->xg, 0, size_t((h->n + 511) & ~int64_t(511)) * h->esz, h->stream) != cudaSuccess)
        rc = sup_fail(h, SUP_ERR_CUDA, "sup_create: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc == SUP_OK) rc = sup_stream_plan(h, h->AT, 0, h->n, false, tab_at, scratch, &h->AT.plan);
    if (rc == SUP_OK) rc = sup_stream_refresh_layout(h);
    if (rc == SUP_OK) rc = sup_setup_wz(h);
    if (rc == SUP_OK && cudaStreamSynchronize(h->stream) != cudaSuccess)
        rc = sup_fail(h, SUP_ERR_CUDA, "sup_create: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc != SUP_OK) {
        memcpy(g_create_error, h->err, sizeof(g_create_error));
        delete h;
        return rc;
    }
    *out = h;
    return SUP_OK;
}

static void drop_graph(sup_ctx* h) {
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    if (h->graph) cudaGraphDestroy(h->graph);
    h->gexec = nullptr;
    h->graph = nullptr;
    h->graph_nodes = 0;
}

extern "C" sup_status sup_destroy(sup_handle h) {
    if (!h) return SUP_OK;
    SUP_ENTER(h);
    cudaStreamSynchronize(h->stream);
    drop_graph(h);
    delete h;
    return SUP_OK;
}

extern "C" sup_status sup_set_blocks(sup_handle h, int n_blocks, const int64_t* block_rowptr, void* workspace,
                                     size_t workspace_bytes, void* scratch, size_t scratch_bytes) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (n_blocks < 1 || !block_rowptr) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_blocks: n_blocks < 1 or NULL block_rowptr");
    if (block_rowptr[0] != 0 || block_rowptr[n_blocks] != h->m)
        return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_blocks: block_rowptr must run from 0 to m");
    for (int t = 0; t < n_blocks; ++t)
        if (block_rowptr[t] > block_rowptr[t + 1]) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_blocks: block_rowptr not monotone");
    size_t need_p = 0, need_s = 0;
    sup_workspace_bytes(SUP_WS_BLOCKS, h->m, h->n, h->nnz, h->dt, n_blocks, &need_p, &need_s);
    if (!workspace || !scratch || workspace_bytes < need_p || scratch_bytes < need_s || !aligned256(workspace) || !aligned256(scratch))
        return sup_fail(h, SUP_ERR_WORKSPACE, "sup_set_blocks: workspace needs %zu + %zu scratch bytes, 256-byte aligned", need_p, need_s);
    drop_graph(h);
    h->n_blocks = 0;
    std::vector<int64_t> ebound(n_blocks + 1);  // A's rowptr at the block boundaries
    for (int t = 0; t <= n_blocks; ++t)
        SUP_CUDA(h, cudaMemcpyAsync(&ebound[t], h->A.rowptr + block_rowptr[t], 8, cudaMemcpyDeviceToHost, h->stream));
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    Bump B{static_cast<char*>(workspace), workspace_bytes, 0, true};
    int32_t* col = static_cast<int32_t*>(B.take(size_t(h->nnz) * 4));
    void* val = B.take(size_t(h->nnz) * h->esz);
    h->d_blk = B.take(size_t(h->m) * h->esz);
    h->pk_atb = h->dt == SUP_F32 ? B.take(size_t(h->nnz) * 8) : nullptr;
    h->ATb.assign(n_blocks, CsrD());
    h->g_bwd_blk.assign(n_blocks, 32);
    h->stream_fwd_blk.assign(n_blocks, StreamPlan());
    h->block_rowptr.assign(block_rowptr, block_rowptr + n_blocks + 1);
    for (int t = 0; t < n_blocks; ++t) {
        int64_t* rowptr_t = static_cast<int64_t*>(B.take(size_t(h->n + 1) * 8));
        if (!B.ok) return sup_fail(h, SUP_ERR_WORKSPACE, "sup_set_blocks: workspace too small");
        sup_status rc = sup_transpose_rows(h, h->A, block_rowptr[t], block_rowptr[t + 1], ebound[t], ebound[t + 1], rowptr_t,
                                           col, val, ebound[t], scratch, scratch_bytes);
        if (rc != SUP_OK) return rc;
        CsrD& T = h->ATb[t];
        T.rows = h->n;
        T.cols = h->m;
        T.nnz = ebound[t + 1] - ebound[t];
        T.rowptr = rowptr_t;
        T.col = col;
        T.val = val;
        T.alloc_nnz = h->nnz;
        T.pk = h->pk_atb;
        h->g_bwd_blk[t] = sup_pick_group(T.nnz, h->n);
        void* tab_f = B.take(sup_stream_table_bytes());
        void* tab_b = B.take(sup_stream_table_bytes());
        if (!B.ok) return sup_fail(h, SUP_ERR_WORKSPACE, "sup_set_blocks: workspace too small");
        rc = sup_stream_plan(h, h->A, block_rowptr[t], block_rowptr[t + 1], true, tab_f, scratch, &h->stream_fwd_blk[t]);
        if (rc == SUP_OK) rc = sup_stream_plan(h, T, 0, h->n, false, tab_b, scratch, &T.plan);
        if (rc != SUP_OK) return rc;
    }
    h->n_blocks = n_blocks;
    sup_status rc = sup_stream_refresh_layout(h);
    if (rc == SUP_OK) rc = sup_setup_block_scaling(h, scratch, scratch_bytes);
    if (rc != SUP_OK) { h->n_blocks = 0; return rc; }
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    return SUP_OK;
}

extern "C" sup_status sup_set_dose_matrix(sup_handle h, const sup_csr* D, void* workspace, size_t workspace_bytes,
                                          void* scratch, size_t scratch_bytes) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!D || !D->rowptr || !D->col || !D->val || D->m <= 0 || D->n != h->n || D->nnz < 0 || D->nnz > 0xfffffffeLL)
        return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_dose_matrix: bad matrix (needs n columns)");
    size_t need_p = 0, need_s = 0;
    sup_workspace_bytes(SUP_WS_DOSE, D->m, D->n, D->nnz, h->dt, 1, &need_p, &need_s);
    if (!workspace || !scratch || workspace_bytes < need_p || scratch_bytes < need_s || !aligned256(workspace) || !aligned256(scratch))
        return sup_fail(h, SUP_ERR_WORKSPACE, "sup_set_dose_matrix: workspace needs %zu + %zu scratch bytes, 256-byte aligned", need_p, need_s);
    drop_graph(h);
    h->has_dose = false;
    CsrD Dm;
    Dm.rows = D->m;
    Dm.cols = D->n;
    Dm.nnz = D->nnz;
    Dm.rowptr = D->rowptr;
    Dm.col = D->col;
    Dm.val = D->val;
    sup_status rc = sup_validate(h, Dm, false, scratch);
    if (rc != SUP_OK) return rc;
    Bump B{static_cast<char*>(workspace), workspace_bytes, 0, true};
    int64_t* rp = static_cast<int64_t*>(B.take(size_t(D->n + 1) * 8));
    int32_t* col = static_cast<int32_t*>(B.take(size_t(D->nnz) * 4));
    void* val = B.take(size_t(D->nnz) * h->esz);
    h->r_dose = B.take(size_t(D->m) * h->esz);
    h->q_dose = B.take(size_t(D->m) * h->esz);
    h->gmean = B.take(size_t(D->n) * h->esz);
    h->gmean_norm2 = static_cast<double*>(B.take(256));
    h->pk_d = h->dt == SUP_F32 ? B.take(size_t(D->nnz) * 8) : nullptr;
    h->pk_dt = h->dt == SUP_F32 ? B.take(size_t(D->nnz) * 8) : nullptr;
    void* tab_d = B.take(sup_stream_table_bytes());
    void* tab_dt = B.take(sup_stream_table_bytes());
    h->gram = h->gram_w = nullptr;
    void *gram = nullptr, *gram_w = nullptr;
    if (sup_gram_applicable(D->n, D->nnz)) {
        gram = B.take(size_t(D->n) * size_t(sup_gram_ld(D->n)) * h->esz);
        gram_w = B.take(size_t(D->n) * h->esz);
    }
    if (!B.ok) return sup_fail(h, SUP_ERR_WORKSPACE, "sup_set_dose_matrix: workspace too small");
    rc = sup_transpose_rows(h, Dm, 0, D->m, 0, D->nnz, rp, col, val, 0, scratch, scratch_bytes);
    if (rc != SUP_OK) return rc;
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    h->D = Dm;
    h->DT.rows = D->n;
    h->DT.cols = D->m;
    h->DT.nnz = D->nnz;
    h->DT.rowptr = rp;
    h->DT.col = col;
    h->DT.val = val;
    h->g_d = sup_pick_group(D->nnz, D->m);
    h->g_dt = sup_pick_group(D->nnz, D->n);
    // the staged product kernels run the dose perturbation's matrix passes: packed copies (plain indices) and plans
    h->D.alloc_nnz = h->DT.alloc_nnz = D->nnz;
    h->D.pk = h->pk_d;
    h->DT.pk = h->pk_dt;
    rc = sup_stream_pack(h, h->D.val, h->D.col, D->nnz, h->pk_d, GMap());
    if (rc == SUP_OK) rc = sup_stream_pack(h, h->DT.val, h->DT.col, D->nnz, h->pk_dt, GMap());
    if (rc == SUP_OK) rc = sup_stream_plan(h, h->D, 0, D->m, true, tab_d, scratch, &h->D.plan);
    if (rc == SUP_OK) rc = sup_stream_plan(h, h->DT, 0, D->n, false, tab_dt, scratch, &h->DT.plan);
    if (rc != SUP_OK) return rc;
    if (gram) {  // the dose objective in n-space: G = D^T D (sup_gram.cu)
        h->gram = gram;
        h->gram_w = gram_w;
        h->gram_ld = sup_gram_ld(D->n);
        rc = sup_gram_build(h);
        if (rc != SUP_OK) {
            h->gram = nullptr;
            return rc;
        }
    }
    h->has_dose = true;
    rc = sup_setup_mean_gradient(h);  // (1/N_S) D^T 1 for f_Mean (Eq. 21), should the matrix be used as a structure's D_S
    if (rc != SUP_OK) return rc;
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    return SUP_OK;
}

extern "C" sup_status sup_set_perturb_mode(sup_handle h, int mode) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (mode != 0 && mode != 1) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_perturb_mode: mode must be 0 (automatic) or 1 (grid kernel)");
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    drop_graph(h);
    h->perturb_mode = mode;
    return SUP_OK;
}

extern "C" sup_status sup_set_dose_mode(sup_handle h, int mode) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (mode != 0 && mode != 1) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_dose_mode: mode must be 0 (automatic) or 1 (matrix passes)");
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    drop_graph(h);
    h->dose_mode = mode;
    return SUP_OK;
}

extern "C" sup_status sup_set_row_mode(sup_handle h, int lanes_forward, int lanes_backward) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    for (int v : {lanes_forward, lanes_backward})
        if (!(v == -2 || v == -1 || v == 0 || v == 1 || v == 2 || v == 4 || v == 8 || v == 16 || v == 32 || v == 64 || v == 128))
            return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_row_mode: lanes must be -2, -1, 0, 1, 2, 4, 8, 16, 32, 64 or 128");
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    drop_graph(h);
    h->use_stream = lanes_forward != -2 && lanes_backward != -2;
    h->lanes_fwd = lanes_forward < 0 ? -1 : lanes_forward;
    h->lanes_bwd = lanes_backward < 0 ? -1 : lanes_backward;
    h->xg_synced = false;
    void* scratch = h->partials;  // 256 bytes are needed
    sup_status rc = sup_stream_plan(h, h->A, 0, h->m, true, h->A.plan.table, scratch, &h->A.plan);
    if (rc == SUP_OK) rc = sup_stream_plan(h, h->AT, 0, h->n, false, h->AT.plan.table, scratch, &h->AT.plan);
    for (int t = 0; rc == SUP_OK && t < h->n_blocks; ++t) {
        rc = sup_stream_plan(h, h->A, h->block_rowptr[t], h->block_rowptr[t + 1], true, h->stream_fwd_blk[t].table, scratch,
                             &h->stream_fwd_blk[t]);
        if (rc == SUP_OK) rc = sup_stream_plan(h, h->ATb[t], 0, h->n, false, h->ATb[t].plan.table, scratch, &h->ATb[t].plan);
    }
    if (rc == SUP_OK && h->has_dose) {
        rc = sup_stream_plan(h, h->D, 0, h->D.rows, true, h->D.plan.table, scratch, &h->D.plan);
        if (rc == SUP_OK) rc = sup_stream_plan(h, h->DT, 0, h->DT.rows, false, h->DT.plan.table, scratch, &h->DT.plan);
    }
    if (rc == SUP_OK) rc = sup_stream_refresh_layout(h);
    if (rc == SUP_OK) SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    return rc;
}

static bool make_tile_map(const int64_t* shape, int64_t size, size_t esz, GMap* out) {
    *out = GMap();
    if (!shape || (shape[0] == 0 && shape[1] == 0)) return true;  // no hint
    if (shape[0] < 1 || shape[1] < 1 || shape[0] * shape[1] != size) return false;
    out->kind = 2;
    out->tw = int(32 / esz);            // one 32-byte sector
    out->th = int(128 / esz) / out->tw;  // 4 sectors = one 128-byte line
    out->C = int(shape[1]);
    out->Rm = int(shape[0] / out->th) * out->th;
    out->Cm = int(shape[1] / out->tw) * out->tw;
    out->ntc = out->Cm / out->tw;
    out->tw_shift = out->tw == 8 ? 3 : 2;  // 32 / esz: 8 (fp32) or 4 (fp64)
    out->th_shift = 2;                     // th = 4
    out->Cmagic = out->C > 1 ? ~0ull / (unsigned long long)out->C + 1ull : 0ull;  // ceil(2^64 / C) (2^64 / C itself for a power of two)
    return true;
}

extern "C" sup_status sup_set_layout(sup_handle h, const int64_t* x_shape, const int64_t* y_shape) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    GMap mx, my;
    if (!make_tile_map(x_shape, h->n, h->esz, &mx)) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_layout: x_shape[0] * x_shape[1] must equal n");
    if (!make_tile_map(y_shape, h->m, h->esz, &my)) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_set_layout: y_shape[0] * y_shape[1] must equal m");
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    drop_graph(h);
    if (mx.kind == 0) mx.kind = 1;  // without a shape: bank swizzle only
    h->xmap = mx;
    h->ymap_req = my;
    sup_status rc = sup_stream_refresh_layout(h);
    if (rc == SUP_OK) SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    return rc;
}

// ---- sweeps ----------------------------------------------------------------------------------------------------
static void enqueue_simultaneous(sup_ctx* h, void* x, double lambda) {
    sup_launch_fwd(h, x, 0, h->m, h->d, &h->A.plan);
    sup_launch_bwd(h, h->AT, h->g_bwd, x, lambda);
}
static void enqueue_block_sweep(sup_ctx* h, void* x, double lambda) {
    for (int t = 0; t < h->n_blocks; ++t) {
        if (h->block_rowptr[t + 1] == h->block_rowptr[t]) continue;
        sup_launch_fwd(h, x, h->block_rowptr[t], h->block_rowptr[t + 1], h->d_blk, &h->stream_fwd_blk[t]);
        sup_launch_bwd(h, h->ATb[t], h->g_bwd_blk[t], x, lambda);
    }
}

static void enqueue_drop(sup_ctx* h, void* x, double lambda) {  // Table A.5: x - lambda Z A^T M c(x)
    sup_launch_fwd(h, x, 0, h->m, h->wT, &h->A.plan);
    sup_launch_bwd(h, h->AT, h->g_bwd, x, lambda, h->zcol);
}
static bool emr_available(const sup_ctx* h) { return h->A.plan.ok && h->AT.plan.ok && (h->colg || h->A.pk) && h->xg; }
static void enqueue_emr(sup_ctx* h, void* x) {  // Table A.5: three matrix passes and one vector update
    double *red_pp = h->red + SUP_STREAM_NBMAX, *red_qq = h->red + 2 * SUP_STREAM_NBMAX;
    sup_launch_fwd(h, x, 0, h->m, h->wT, &h->A.plan);                   // y = M c(x)
    sup_launch_stream_plain_AT(h, h->g2, 1.0, red_pp);                 // p = A^T y (in x's gather layout), sum p^2
    sup_launch_stream_plain_A(h, h->g2, h->y, 1.0, h->wT, red_qq);     // q = A p (over y, no longer needed), sum w q^2
    sup_launch_emr_update(h, red_pp, h->AT.plan.nb, red_qq, h->A.plan.nb, h->g2, x);
}

static sup_status check_lambda(sup_ctx* h, double lambda) {
    if (!(lambda >= 0.0 && lambda <= 2.0)) return sup_fail(h, SUP_ERR_INVALID_ARG, "lambda must be in [0,2] (PAPER.md:L44)");
    return SUP_OK;
}

extern "C" sup_status sup_project_simultaneous(sup_handle h, void* x, double lambda, int n_sweeps) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || n_sweeps < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_project_simultaneous: NULL x or n_sweeps < 0");
    if (check_lambda(h, lambda) != SUP_OK) return SUP_ERR_INVALID_ARG;
    h->xg_synced = false;  // x comes from the caller
    for (int s = 0; s < n_sweeps; ++s) enqueue_simultaneous(h, x, lambda);
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

extern "C" sup_status sup_forward_violation(sup_handle h, const void* x) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_forward_violation: NULL x");
    h->xg_synced = false;
    sup_launch_fwd(h, x, 0, h->m, h->d, &h->A.plan);
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

extern "C" sup_status sup_backproject_update(sup_handle h, void* x, double lambda) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_backproject_update: NULL x");
    if (check_lambda(h, lambda) != SUP_OK) return SUP_ERR_INVALID_ARG;
    sup_launch_bwd(h, h->AT, h->g_bwd, x, lambda);
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

// ---- the two halves of a ROW-SHARDED sweep: each GPU holds a block of rows of A and a replica of x ------------
template <typename T>
__global__ void __launch_bounds__(SUP_THREADS) k_apply_update(T* __restrict__ x, const T* __restrict__ u, const T* __restrict__ lo,
                                                             const T* __restrict__ hi, T lambda, int64_t n, T* __restrict__ xg, const GMap xmap) {
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n; j += int64_t(gridDim.x) * blockDim.x) {
        T t = x[j] - lambda * u[j];  // Eq. 3
        t = t < lo[j] ? lo[j] : t;   // box (L427)
        t = t > hi[j] ? hi[j] : t;
        x[j] = t;
        if (xg) xg[sup_gmap(xmap, int(j))] = t;
    }
}

extern "C" sup_status sup_backproject_partial(sup_handle h, void* u, double scale) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!u) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_backproject_partial: NULL u");
    if (!h->AT.plan.ok) return sup_fail(h, SUP_ERR_STATE, "sup_backproject_partial needs the staged product kernels (sup_set_row_mode)");
    sup_launch_staged(h, 2, h->AT.plan, h->AT, h->y, nullptr, nullptr, nullptr, u, nullptr, scale, GMap(), h->ymap.kind == 2, nullptr);
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

extern "C" sup_status sup_apply_update(sup_handle h, void* x, const void* u, double lambda) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || !u) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_apply_update: NULL x or u");
    if (check_lambda(h, lambda) != SUP_OK) return SUP_ERR_INVALID_ARG;
    const int grid = sup_grid_for(h->n, SUP_THREADS, h->num_sms * 4);
    void* mirror = sup_stream_forward_uses_xg(h) ? h->xg : nullptr;
    if (h->dt == SUP_F32)
        k_apply_update<float><<<grid, SUP_THREADS, 0, h->stream>>>(static_cast<float*>(x), static_cast<const float*>(u), static_cast<const float*>(h->lo),
                                                                   static_cast<const float*>(h->hi), float(lambda), h->n, static_cast<float*>(mirror), h->xmap);
    else
        k_apply_update<double><<<grid, SUP_THREADS, 0, h->stream>>>(static_cast<double*>(x), static_cast<const double*>(u), static_cast<const double*>(h->lo),
                                                                    static_cast<const double*>(h->hi), lambda, h->n, static_cast<double*>(mirror), h->xmap);
    h->launches++;
    h->xg_synced = mirror != nullptr;
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

extern "C" sup_status sup_project_drop(sup_handle h, void* x, double lambda, int n_sweeps) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || n_sweeps < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_project_drop: NULL x or n_sweeps < 0");
    if (check_lambda(h, lambda) != SUP_OK) return SUP_ERR_INVALID_ARG;
    h->xg_synced = false;
    for (int s = 0; s < n_sweeps; ++s) enqueue_drop(h, x, lambda);
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

extern "C" sup_status sup_project_emr(sup_handle h, void* x, int n_sweeps) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || n_sweeps < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_project_emr: NULL x or n_sweeps < 0");
    if (!emr_available(h)) return sup_fail(h, SUP_ERR_STATE, "sup_project_emr needs the staged product kernels (sup_set_row_mode)");
    h->xg_synced = false;
    for (int s = 0; s < n_sweeps; ++s) enqueue_emr(h, x);
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

extern "C" sup_status sup_block_iterative(sup_handle h, void* x, double lambda, int n_sweeps) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || n_sweeps < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_block_iterative: NULL x or n_sweeps < 0");
    if (h->n_blocks < 1) return sup_fail(h, SUP_ERR_STATE, "sup_block_iterative: call sup_set_blocks first");
    if (check_lambda(h, lambda) != SUP_OK) return SUP_ERR_INVALID_ARG;
    h->xg_synced = false;
    for (int s = 0; s < n_sweeps; ++s) enqueue_block_sweep(h, x, lambda);
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

// ---- perturbation phase alone ----------------------------------------------------------------------------------
static sup_status check_step(sup_ctx* h, int N, double beta0, double a) {
    if (N < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "N must be >= 0");
    if (!(beta0 >= 0.0) || isinf(beta0)) return sup_fail(h, SUP_ERR_INVALID_ARG, "beta0 must be finite and >= 0");
    if (!(a > 0.0 && a < 1.0)) return sup_fail(h, SUP_ERR_INVALID_ARG, "a must be in (0,1) (PAPER.md:L99)");
    return SUP_OK;
}

// dims = {nz, ny, nx} of the objective's view of x (0 where unused)
static sup_status check_objective(sup_ctx* h, int kind, const int64_t* shape, int64_t* dims) {
    dims[0] = dims[1] = dims[2] = 0;
    switch (kind) {
        case SUP_OBJ_NONE:
        case SUP_OBJ_TV1D: return SUP_OK;
        case SUP_OBJ_TV2D:
            if (!shape || shape[0] < 1 || shape[1] < 1 || shape[0] * shape[1] != h->n)
                return sup_fail(h, SUP_ERR_INVALID_ARG, "TV2D needs shape = {ny, nx} with ny*nx == n");
            dims[1] = shape[0];
            dims[2] = shape[1];
            return SUP_OK;
        case SUP_OBJ_TV3D:
            if (!shape || shape[0] < 1 || shape[1] < 1 || shape[2] < 1 || shape[0] * shape[1] * shape[2] != h->n)
                return sup_fail(h, SUP_ERR_INVALID_ARG, "TV3D needs shape = {nz, ny, nx} with nz*ny*nx == n");
            dims[0] = shape[0];
            dims[1] = shape[1];
            dims[2] = shape[2];
            return SUP_OK;
        case SUP_OBJ_DOSE:
        case SUP_OBJ_MEAN:
            if (!h->has_dose) return sup_fail(h, SUP_ERR_STATE, "dose / mean objective: call sup_set_dose_matrix first");
            return SUP_OK;
    }
    return sup_fail(h, SUP_ERR_INVALID_ARG, "unknown objective kind %d", kind);
}

static sup_status read_state(sup_ctx* h, sup_state* out) {
    DevState s;
    SUP_CUDA(h, cudaMemcpyAsync(&s, h->state, sizeof(DevState), cudaMemcpyDeviceToHost, h->stream));
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    out->ell = s.ell;
    out->k = s.k;
    out->n_trials = s.n_trials;
    out->n_decisions = s.n_dec;
    out->warn = s.warn;
    out->fault = s.fault;
    out->f = s.f;
    out->n_done = s.n_done;
    out->stop_reason = s.stop_reason;
    out->step = s.step;
    out->f_ref = s.f_ref;
    return SUP_OK;
}

extern "C" sup_status sup_get_state(sup_handle h, sup_state* out) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!out) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_get_state: NULL out");
    sup_status rc = read_state(h, out);
    if (rc != SUP_OK) return rc;
    if (out->fault & 1) return sup_fail(h, SUP_ERR_CUDA, "device-side grid barrier timed out");
    if (out->fault & 2) return sup_fail(h, SUP_ERR_NONFINITE, "non-finite objective value");
    return SUP_OK;
}

// Eq. 11's rule (A-30) is built for the objectives whose phase evaluates f and g in every step
static sup_status check_adaptive(sup_ctx* h, int objective, double f_ref, double shrink) {
    if (objective != SUP_OBJ_TV1D && objective != SUP_OBJ_TV2D && objective != SUP_OBJ_TV3D && objective != SUP_OBJ_DOSE)
        return sup_fail(h, SUP_ERR_INVALID_ARG, "the adaptive step rule (Eq. 11) is available for TV and dose objectives");
    if (!(shrink > 0.0 && shrink <= 1.0)) return sup_fail(h, SUP_ERR_INVALID_ARG, "f_ref_shrink must be in (0, 1]");
    if (!std::isfinite(f_ref)) return sup_fail(h, SUP_ERR_INVALID_ARG, "f_ref must be finite");
    return SUP_OK;
}

extern "C" sup_status sup_perturb_adaptive(sup_handle h, void* x, int objective, const int64_t* shape, int N, double* f_ref, double shrink) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || !f_ref || N < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_perturb_adaptive: NULL x / f_ref or N < 0");
    sup_status rc = check_adaptive(h, objective, *f_ref, shrink);
    if (rc != SUP_OK) return rc;
    int64_t dims[3];
    rc = check_objective(h, objective, shape, dims);
    if (rc != SUP_OK) return rc;
    sup_launch_begin_run(h, 0, 0, 1.0, 0, *f_ref);
    if (N > 0) {
        PerturbParams pp = {objective, dims[0], dims[1], dims[2], N, 0.0, 1.0, SUP_STEP_PER_TRIAL, nullptr, nullptr, 0, 0, false, SUP_RULE_ADAPTIVE, shrink};
        rc = sup_launch_perturb(h, x, pp);
        if (rc != SUP_OK) return rc;
    }
    sup_state s;
    rc = sup_get_state(h, &s);
    if (rc != SUP_OK) return rc;
    *f_ref = s.f_ref;
    return SUP_OK;
}

static sup_status perturb_alone(sup_ctx* h, void* x, int kind, const int64_t* shape, int N, double beta0, double a, int64_t* ell) {
    if (!x || !ell) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_perturb: NULL x or ell");
    if (check_step(h, N, beta0, a) != SUP_OK) return SUP_ERR_INVALID_ARG;
    int64_t dims[3];
    sup_status rc = check_objective(h, kind, shape, dims);
    if (rc != SUP_OK) return rc;
    sup_launch_begin_run(h, *ell, 0, a);
    if (N > 0) {
        PerturbParams pp = {kind, dims[0], dims[1], dims[2], N, beta0, a, SUP_STEP_PER_TRIAL, nullptr, nullptr, 0, 0, false};
        rc = sup_launch_perturb(h, x, pp);
        if (rc != SUP_OK) return rc;
    }
    sup_state s;
    rc = sup_get_state(h, &s);
    if (rc != SUP_OK) return rc;
    *ell = s.ell;
    return SUP_OK;
}

extern "C" sup_status sup_perturb_tv(sup_handle h, void* x, int dims, const int64_t* shape, int N, double beta0, double a,
                                     int64_t* ell) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (dims < 1 || dims > 3) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_perturb_tv: dims must be 1, 2 or 3");
    if (dims == 1 && shape && shape[0] != h->n) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_perturb_tv: shape[0] != n");
    return perturb_alone(h, x, dims == 3 ? SUP_OBJ_TV3D : (dims == 2 ? SUP_OBJ_TV2D : SUP_OBJ_TV1D), shape, N, beta0, a, ell);
}

extern "C" sup_status sup_perturb_dose(sup_handle h, void* x, int N, double beta0, double a, int64_t* ell) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    return perturb_alone(h, x, SUP_OBJ_DOSE, nullptr, N, beta0, a, ell);
}

extern "C" sup_status sup_perturb_mean(sup_handle h, void* x, int N, double beta0, double a, int64_t* ell) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    return perturb_alone(h, x, SUP_OBJ_MEAN, nullptr, N, beta0, a, ell);
}

// ---- Algorithm 1 -----------------------------------------------------------------------------------------------
struct RunPlan {
    void* x;
    int N;
    double beta0, a;
    sup_options o;
    int64_t dims[3];  // {nz, ny, nx} of the objective
};

static bool run_perturbed(const RunPlan& P) { return P.N > 0 && P.o.objective != SUP_OBJ_NONE; }
// the basic simultaneous sweep gets the proximity of its iterate for free from the forward product's epilogue
static bool run_free_prox(const sup_ctx* h, const RunPlan& P) {
    return !run_perturbed(P) && P.o.algorithm == SUP_ALG_DEFAULT && !P.o.block_iterative && h->A.plan.ok &&
           ((P.o.trace_mode && P.o.trace) || P.o.stop_enabled);
}

// f(x) into state->scalar_out
static void enqueue_objective(sup_ctx* h, const RunPlan& P) {
    double* slot = reinterpret_cast<double*>(reinterpret_cast<char*>(h->state) + offsetof(DevState, scalar_out));
    sup_launch_objective(h, P.x, P.o.objective, P.dims[0], P.dims[1], P.dims[2], slot);
}

// (P, f) of the current x for the trace / the stopping rule: one forward pass whose epilogue reduces sum c_i y_i (Eq. 12,
// p = 2) -- or the plain proximity kernel when the staged kernels are off -- and the objective value; then the closing kernel
static void enqueue_measure_and_close(sup_ctx* h, const RunPlan& P, int mode) {
    int np = 0;
    if (h->A.plan.ok) {
        sup_launch_fwd(h, P.x, 0, h->m, h->d, &h->A.plan, h->red);
        np = h->A.plan.nb;
    } else {
        double* slot = reinterpret_cast<double*>(reinterpret_cast<char*>(h->state) + offsetof(DevState, prox_cur));
        sup_launch_proximity(h, P.x, 0, 2.0, slot);
    }
    enqueue_objective(h, P);
    sup_launch_close_sweep(h, P.o.trace, h->red, np, mode, 1, run_perturbed(P), P.o);
}

static sup_status enqueue_superiorized_sweep(sup_ctx* h, const RunPlan& P) {
    if (run_perturbed(P)) {
        PerturbParams pp = {P.o.objective, P.dims[0], P.dims[1], P.dims[2], P.N, P.beta0, P.a, P.o.step_policy, P.o.decisions,
                            P.o.decision_f, P.o.decisions_cap, P.o.n_restart, true, P.o.step_rule, P.o.f_ref_shrink};
        sup_status rc = sup_launch_perturb(h, P.x, pp);
        if (rc != SUP_OK) return rc;
        h->xg_synced = sup_stream_forward_uses_xg(h);  // the perturbation kernel wrote the moved x to the gather mirror too
    }
    const bool measure = (P.o.trace_mode && P.o.trace) || P.o.stop_enabled;
    if (run_free_prox(h, P)) {
        sup_launch_fwd(h, P.x, 0, h->m, h->d, &h->A.plan, h->red);
        sup_launch_close_sweep(h, P.o.trace, h->red, h->A.plan.nb, 2, 0, 0, P.o);  // P(x^k): trace row k-1, rule, or P^0
        sup_launch_bwd(h, h->AT, h->g_bwd, P.x, P.o.lambda);
        sup_launch_close_sweep(h, P.o.trace, nullptr, 0, 3, 0, 0, P.o);
        return SUP_OK;
    }
    if (P.o.algorithm == SUP_ALG_DROP) enqueue_drop(h, P.x, P.o.lambda);
    else if (P.o.algorithm == SUP_ALG_EMR) enqueue_emr(h, P.x);
    else if (P.o.block_iterative) enqueue_block_sweep(h, P.x, P.o.lambda);
    else enqueue_simultaneous(h, P.x, P.o.lambda);
    if (measure) enqueue_measure_and_close(h, P, 0);
    else sup_launch_close_sweep(h, P.o.trace, nullptr, 0, 3, 0, 0, P.o);
    return SUP_OK;
}

static sup_status run_superiorize(sup_ctx* h, void* x, int n_iter, int N, double beta0, double a, const sup_options* opt) {
    if (!x || !opt || n_iter < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_superiorize: NULL x/opt or n_iter < 0");
    if (check_step(h, N, beta0, a) != SUP_OK || check_lambda(h, opt->lambda) != SUP_OK) return SUP_ERR_INVALID_ARG;
    if (opt->step_policy != SUP_STEP_PER_TRIAL && opt->step_policy != SUP_STEP_PER_SWEEP)
        return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_superiorize: unknown step policy");
    if (opt->block_iterative && h->n_blocks < 1) return sup_fail(h, SUP_ERR_STATE, "sup_superiorize: call sup_set_blocks first");
    if ((opt->decisions || opt->decision_f) && opt->decisions_cap < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "decisions_cap < 0");
    if (opt->n_restart < 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "n_restart < 0");
    if (opt->ell0 < 0 || opt->ell0 > 10000000) return sup_fail(h, SUP_ERR_INVALID_ARG, "ell0 must be in [0, 1e7] (a^l is formed by l multiplications, A-20)");
    if (opt->algorithm != SUP_ALG_DEFAULT && opt->algorithm != SUP_ALG_DROP && opt->algorithm != SUP_ALG_EMR)
        return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_superiorize: unknown algorithm");
    if (opt->algorithm != SUP_ALG_DEFAULT && opt->block_iterative)
        return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_superiorize: DROP / EMR are simultaneous operators (block_iterative must be 0)");
    if (opt->algorithm == SUP_ALG_EMR && !emr_available(h))
        return sup_fail(h, SUP_ERR_STATE, "EMR needs the staged product kernels (sup_set_row_mode)");
    if (opt->stop_enabled && (opt->n_consec < 1 || !(opt->dprox_tol >= 0.0) || !(opt->dobj_tol >= 0.0)))
        return sup_fail(h, SUP_ERR_INVALID_ARG, "stopping rule: n_consec >= 1 and non-negative thresholds are needed");
    if (opt->step_rule != SUP_RULE_POWER && opt->step_rule != SUP_RULE_ADAPTIVE) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_superiorize: unknown step rule");
    if (opt->step_rule == SUP_RULE_ADAPTIVE && N > 0 && opt->objective != SUP_OBJ_NONE) {
        sup_status ra = check_adaptive(h, opt->objective, opt->f_ref, opt->f_ref_shrink);
        if (ra != SUP_OK) return ra;
        if (opt->n_restart > 0) return sup_fail(h, SUP_ERR_INVALID_ARG, "restarts belong to the power law (the adaptive rule has no exponent)");
    }
    RunPlan P;
    P.x = x;
    P.N = N;
    P.beta0 = beta0;
    P.a = a;
    P.o = *opt;
    sup_status rc = check_objective(h, opt->objective, opt->shape, P.dims);
    if (rc != SUP_OK) return rc;
    sup_launch_begin_run(h, opt->ell0, opt->k0, a, n_iter, opt->f_ref);
    h->xg_synced = false;
    h->stop_ptr = opt->stop_enabled ? &h->state->stop : nullptr;
    struct StopPtrReset {
        sup_ctx* h;
        ~StopPtrReset() { h->stop_ptr = nullptr; }
    } stop_ptr_reset{h};
    if (opt->stop_enabled && n_iter > 0 && !run_free_prox(h, P)) enqueue_measure_and_close(h, P, 1);  // P^0, f^0

    bool graph = opt->use_graph && h->stream != nullptr && !h->graph_failed && n_iter > 1;
    if (graph) {
        sup_ctx::GraphKey key;
        key.x = x;
        key.N = N;
        key.objective = opt->objective;
        key.block = opt->block_iterative;
        key.policy = opt->step_policy;
        key.trace_mode = opt->trace_mode;
        key.beta0 = beta0;
        key.a = a;
        key.lambda = opt->lambda;
        key.s0 = P.dims[1];
        key.s1 = P.dims[2];
        key.s2 = P.dims[0];
        key.trace = opt->trace;
        key.dec = opt->decisions;
        key.decf = opt->decision_f;
        key.cap = opt->decisions_cap;
        key.n_restart = opt->n_restart;
        key.algorithm = opt->algorithm;
        key.stop = opt->stop_enabled;
        key.tols[0] = opt->prox_tol;
        key.tols[1] = opt->dprox_tol;
        key.tols[2] = opt->dobj_tol;
        key.n_consec = opt->n_consec;
        key.step_rule = opt->step_rule;
        key.shrink = opt->f_ref_shrink;
        if (!h->gexec || !(key == h->gkey)) {
            drop_graph(h);
            const int64_t launches_before = h->launches;
            cudaError_t e = cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal);
            if (e == cudaSuccess) {
                rc = enqueue_superiorized_sweep(h, P);
                cudaGraph_t gr = nullptr;
                e = cudaStreamEndCapture(h->stream, &gr);
                if (rc == SUP_OK && e == cudaSuccess && gr) {
                    h->graph = gr;
                    e = cudaGraphInstantiate(&h->gexec, gr, 0);
                    size_t nn = 0;
                    if (e == cudaSuccess) cudaGraphGetNodes(gr, nullptr, &nn);
                    h->graph_nodes = int(nn);
                } else if (gr) {
                    cudaGraphDestroy(gr);
                }
            }
            h->launches = launches_before;
            if (e != cudaSuccess || rc != SUP_OK || !h->gexec) {
                cudaGetLastError();
                drop_graph(h);
                h->graph_failed = true;  // e.g. cooperative launch not capturable: fall back to direct launches
                graph = false;
            } else {
                h->gkey = key;
            }
        }
    }
    for (int it = 0; it < n_iter; ++it) {
        if (graph) {
            SUP_CUDA(h, cudaGraphLaunch(h->gexec, h->stream));
            h->launches += h->graph_nodes;
        } else {
            rc = enqueue_superiorized_sweep(h, P);
            if (rc != SUP_OK) return rc;
        }
    }
    if (n_iter > 0 && run_free_prox(h, P) && P.o.trace_mode && P.o.trace) {  // proximity of the final iterate for the last trace row
        sup_launch_fwd(h, P.x, 0, h->m, h->d, &h->A.plan, h->red);
        sup_launch_close_sweep(h, P.o.trace, h->red, h->A.plan.nb, 4, 0, 0, P.o);
    }
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

extern "C" sup_status sup_superiorize(sup_handle h, void* x, int n_iter, int N, double beta0, double a, const sup_options* opt) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    return run_superiorize(h, x, n_iter, N, beta0, a, opt);
}

extern "C" sup_status sup_superiorize_host(sup_handle h, void* x_host, int n_iter, int N, double beta0, double a,
                                           const sup_options* opt) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x_host) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_superiorize_host: NULL x");
    const size_t bytes = size_t(h->n) * h->esz;
    SUP_CUDA(h, cudaMemcpyAsync(h->xdev, x_host, bytes, cudaMemcpyHostToDevice, h->stream));
    sup_status rc = run_superiorize(h, h->xdev, n_iter, N, beta0, a, opt);
    if (rc != SUP_OK) return rc;
    SUP_CUDA(h, cudaMemcpyAsync(x_host, h->xdev, bytes, cudaMemcpyDeviceToHost, h->stream));
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    return SUP_OK;
}

// ---- scalars -----------------------------------------------------------------------------------------------------
static sup_status fetch_scalar(sup_ctx* h, double* out) {
    const double* slot = reinterpret_cast<const double*>(reinterpret_cast<const char*>(h->state) + offsetof(DevState, scalar_out));
    SUP_CUDA(h, cudaMemcpyAsync(out, slot, 8, cudaMemcpyDeviceToHost, h->stream));
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    if (isnan(*out)) return sup_fail(h, SUP_ERR_NONFINITE, "result is NaN");
    return SUP_OK;
}

extern "C" sup_status sup_proximity(sup_handle h, const void* x, int mode, double p, double* out) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || !out || mode < 0 || mode > 2) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_proximity: NULL x/out or mode not in {0,1,2}");
    if (mode == 1 && !(p > 0.0)) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_proximity: p must be > 0");
    double* slot = reinterpret_cast<double*>(reinterpret_cast<char*>(h->state) + offsetof(DevState, scalar_out));
    sup_launch_proximity(h, x, mode, p, slot);
    return fetch_scalar(h, out);
}

extern "C" sup_status sup_objective(sup_handle h, const void* x, int kind, const int64_t* shape, double* out) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    if (!x || !out) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_objective: NULL x or out");
    int64_t dims[3];
    sup_status rc = check_objective(h, kind, shape, dims);
    if (rc != SUP_OK) return rc;
    double* slot = reinterpret_cast<double*>(reinterpret_cast<char*>(h->state) + offsetof(DevState, scalar_out));
    sup_launch_objective(h, x, kind, dims[0], dims[1], dims[2], slot);
    return fetch_scalar(h, out);
}

extern "C" sup_status sup_get_derived(sup_handle h, int which, void* dst, size_t dst_bytes) {
    if (!h) return SUP_ERR_INVALID_ARG;
    SUP_ENTER(h);
    const void* src = nullptr;
    size_t bytes = 0;
    switch (which) {
        case 0: src = h->d; bytes = size_t(h->m) * h->esz; break;
        case 1: src = h->AT.rowptr; bytes = size_t(h->n + 1) * 8; break;
        case 2: src = h->AT.col; bytes = size_t(h->nnz) * 4; break;
        case 3: src = h->AT.val; bytes = size_t(h->nnz) * h->esz; break;
        case 5: src = h->y; bytes = size_t(h->m) * h->esz; break;  // y = D c(x) of the last forward product
        default: return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_get_derived: unknown array");
    }
    if (!dst || dst_bytes < bytes) return sup_fail(h, SUP_ERR_INVALID_ARG, "sup_get_derived: dst too small (%zu needed)", bytes);
    if (which == 5 && h->ymap.kind != 0) sup_launch_unmap(h, h->y, dst, h->m, h->ymap);  // y is kept in its gather layout
    else SUP_CUDA(h, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, h->stream));
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    return SUP_OK;
}
