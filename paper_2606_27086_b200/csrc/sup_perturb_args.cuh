// sup_perturb_args.cuh -- the argument block of the perturbation kernels (sup_perturb.cu, sup_perturb_small.cu)
#pragma once
#include "sup_internal.cuh"

template <typename T>
struct PArgs {
    T* x;
    T* g;
    T* x2;  // second iterate / gradient buffers (TV objectives: an accepted step is applied inside the next gradient pass)
    T* g2;
    int64_t n, nz, ny, nx;
    T* xg;      // gather mirror of x kept by the product kernels (NULL: none): written together with the final iterate
    GMap xmap;
    int N;
    double beta0, a;
    int policy;
    long long n_restart;
    int step_rule;  // sup_step_rule
    double shrink;  // adaptive rule (A-30)
    DevState* st;
    double* partials;  // [2][SUP_MAX_PARTIALS]
    int8_t* decisions;
    double* decision_f;
    int64_t cap;
    // dose
    int64_t md;
    const int64_t* d_rowptr;
    const int32_t* d_col;
    const T* d_val;
    const int64_t* dt_rowptr;
    const int32_t* dt_col;
    const T* dt_val;
    T* r;
    T* q;  // [md]: D g of the current reduction step (dose objective)
    int g_d, g_dt;
};

template <typename T>
inline PArgs<T> sup_make_perturb_args(sup_ctx* h, void* x, const PerturbParams& pp) {
    PArgs<T> A;
    A.x = static_cast<T*>(x);
    A.g = static_cast<T*>(h->g);
    A.x2 = static_cast<T*>(h->x2);
    A.g2 = static_cast<T*>(h->g2);
    A.n = h->n;
    A.nz = pp.nz;
    A.ny = pp.ny;
    A.nx = pp.nx;
    A.xg = pp.write_mirror && sup_stream_forward_uses_xg(h) ? static_cast<T*>(h->xg) : nullptr;
    A.xmap = h->xmap;
    A.N = pp.N;
    A.beta0 = pp.beta0;
    A.a = pp.a;
    A.policy = pp.policy;
    A.step_rule = pp.step_rule;
    A.shrink = pp.shrink;
    A.n_restart = pp.n_restart;
    A.st = h->state;
    A.partials = h->partials;
    A.decisions = pp.decisions;
    A.decision_f = pp.decision_f;
    A.cap = pp.cap;
    A.md = h->D.rows;
    A.d_rowptr = h->D.rowptr;
    A.d_col = h->D.col;
    A.d_val = static_cast<const T*>(h->D.val);
    A.dt_rowptr = h->DT.rowptr;
    A.dt_col = h->DT.col;
    A.dt_val = static_cast<const T*>(h->DT.val);
    A.r = static_cast<T*>(h->r_dose);
    A.q = static_cast<T*>(h->q_dose);
    A.g_d = h->g_d;
    A.g_dt = h->g_dt;
    return A;
}
