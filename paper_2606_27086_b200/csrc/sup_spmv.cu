// sup_spmv.cu -- S1-S4 of the hot path.
//   S1+S2  k_fwd : r_i = <a_i, x>, hyperslab violation c_i (Eq. 2 on each face, L38-42; Eq. 20),
//                  y_i = d_i c_i with d_i = w_i/||a_i||^2 (L608).  r is never written.
//   S3     k_bwd : u_j = sum_i a_ij y_i over row j of the explicit A^T, x_j <- clip(x_j - lambda u_j) (Eq. 3; box L427).
//   S4     k_prox: the three proximity functions (Eq. 5, Eq. 12, Eq. 13).
// Both products are atomic-free row gathers: a group of G lanes (G a power of two chosen from the mean row
// length) owns one row, streams its values/indices with coalesced loads and reduces with warp shuffles.
#include <math.h>

#include "sup_internal.cuh"

template <typename T>
__device__ __forceinline__ T ld_stream(const T* p) {  // streamed once: read-only path, do not keep in L1
    return __ldcs(p);
}

// dot product of CSR row [s, e) with the dense vector v, computed by the G lanes of a group (lane gl of G)
template <typename T>
__device__ __forceinline__ T group_row_dot(const T* __restrict__ val, const int32_t* __restrict__ col, int64_t s, int64_t e,
                                           const T* __restrict__ v, int gl, int G) {
    T a0 = T(0), a1 = T(0), a2 = T(0), a3 = T(0);
    int64_t k = s + gl;
    const int64_t G4 = 4 * int64_t(G);
    for (; k + 3 * int64_t(G) < e; k += G4) {
        const int c0 = ld_stream(col + k), c1 = ld_stream(col + k + G), c2 = ld_stream(col + k + 2 * G),
                  c3 = ld_stream(col + k + 3 * G);
        const T v0 = ld_stream(val + k), v1 = ld_stream(val + k + G), v2 = ld_stream(val + k + 2 * G),
                v3 = ld_stream(val + k + 3 * G);
        a0 += v0 * __ldg(v + c0);
        a1 += v1 * __ldg(v + c1);
        a2 += v2 * __ldg(v + c2);
        a3 += v3 * __ldg(v + c3);
    }
    for (; k < e; k += G) a0 += ld_stream(val + k) * __ldg(v + ld_stream(col + k));
    T acc = (a0 + a1) + (a2 + a3);
    for (int o = G >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o, G);
    return acc;
}

template <typename T>
__device__ __forceinline__ T violation(T r, T lb, T ub) {  // Eq. 2 on each face of lb <= r <= ub; at most one is violated
    return r > ub ? r - ub : (r < lb ? r - lb : T(0));
}

template <typename T>
__global__ void __launch_bounds__(SUP_THREADS)
    k_fwd(int64_t r0, int64_t r1, const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
          const T* __restrict__ val, const T* __restrict__ x, const T* __restrict__ lb, const T* __restrict__ ub,
          const T* __restrict__ d, T* __restrict__ y, int G, const int* __restrict__ stop) {
    if (stop && *stop) return;
    const int gl = threadIdx.x % G;
    const int64_t i = r0 + (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) / G;
    const bool valid = i < r1;
    const int64_t s = valid ? rowptr[i] : 0, e = valid ? rowptr[i + 1] : 0;
    const T r = group_row_dot(val, col, s, e, x, gl, G);
    if (valid && gl == 0) y[i] = d[i] * violation(r, lb[i], ub[i]);
}

template <typename T>
__global__ void __launch_bounds__(SUP_THREADS)
    k_bwd(int64_t n, const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col, const T* __restrict__ val,
          const T* __restrict__ y, const T* __restrict__ lo, const T* __restrict__ hi, T lambda, T* __restrict__ x,
          T* __restrict__ xg, int G, const GMap xmap, const T* __restrict__ zscale, const int* __restrict__ stop) {
    if (stop && *stop) return;
    const int gl = threadIdx.x % G;
    const int64_t j = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) / G;
    const bool valid = j < n;
    const int64_t s = valid ? rowptr[j] : 0, e = valid ? rowptr[j + 1] : 0;
    const T u = group_row_dot(val, col, s, e, y, gl, G);
    if (valid && gl == 0) {
        T t = x[j] - lambda * ((zscale ? zscale[j] : T(1)) * u);  // Eq. 3 (zscale: DROP's 1/nnz(A_:,j))
        t = t < lo[j] ? lo[j] : t;  // box, un-relaxed (A-2)
        t = t > hi[j] ? hi[j] : t;
        x[j] = t;
        if (xg) xg[sup_gmap(xmap, int(j))] = t;  // gather mirror read by the staged forward product (sup_stream.cu)
    }
}

void sup_launch_fwd(sup_ctx* h, const void* x, int64_t r0, int64_t r1, const void* dscale, const StreamPlan* rp, double* red_out) {
    const int G = h->g_fwd;
    const int64_t rows = r1 - r0;
    if (rows <= 0) return;
    if (rp && rp->ok) {
        sup_launch_stream_fwd(h, *rp, x, dscale, red_out);
        return;
    }
    const unsigned grid = unsigned((rows * G + SUP_THREADS - 1) / SUP_THREADS);
    if (h->dt == SUP_F32)
        k_fwd<float><<<grid, SUP_THREADS, 0, h->stream>>>(
            r0, r1, h->A.rowptr, h->A.col, static_cast<const float*>(h->A.val), static_cast<const float*>(x),
            static_cast<const float*>(h->lb), static_cast<const float*>(h->ub), static_cast<const float*>(dscale),
            static_cast<float*>(h->y), G, h->stop_ptr);
    else
        k_fwd<double><<<grid, SUP_THREADS, 0, h->stream>>>(
            r0, r1, h->A.rowptr, h->A.col, static_cast<const double*>(h->A.val), static_cast<const double*>(x),
            static_cast<const double*>(h->lb), static_cast<const double*>(h->ub), static_cast<const double*>(dscale),
            static_cast<double*>(h->y), G, h->stop_ptr);
    h->launches++;
}

void sup_launch_bwd(sup_ctx* h, const CsrD& AT, int G, void* x, double lambda, const void* zscale) {
    if (AT.plan.ok) {
        sup_launch_stream_bwd(h, AT, AT.plan, x, lambda, zscale);
        return;
    }
    const unsigned grid = unsigned((AT.rows * G + SUP_THREADS - 1) / SUP_THREADS);
    void* mirror = sup_stream_forward_uses_xg(h) ? h->xg : nullptr;
    h->xg_synced = mirror != nullptr;
    if (h->dt == SUP_F32)
        k_bwd<float><<<grid, SUP_THREADS, 0, h->stream>>>(
            AT.rows, AT.rowptr, AT.col, static_cast<const float*>(AT.val), static_cast<const float*>(h->y),
            static_cast<const float*>(h->lo), static_cast<const float*>(h->hi), float(lambda), static_cast<float*>(x),
            static_cast<float*>(mirror), G, h->xmap, static_cast<const float*>(zscale), h->stop_ptr);
    else
        k_bwd<double><<<grid, SUP_THREADS, 0, h->stream>>>(
            AT.rows, AT.rowptr, AT.col, static_cast<const double*>(AT.val), static_cast<const double*>(h->y),
            static_cast<const double*>(h->lo), static_cast<const double*>(h->hi), lambda, static_cast<double*>(x),
            static_cast<double*>(mirror), G, h->xmap, static_cast<const double*>(zscale), h->stop_ptr);
    h->launches++;
}

// ---- S4 proximity ------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(SUP_THREADS)
    k_prox(int64_t m, const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col, const T* __restrict__ val,
           const T* __restrict__ x, const T* __restrict__ lb, const T* __restrict__ ub, const double* __restrict__ w,
           const double* __restrict__ invnorm, int mode, double p, double* __restrict__ partials, int G) {
    __shared__ double ws[SUP_THREADS / 32];
    const int gl = threadIdx.x % G, lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t gid = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) / G;
    const int64_t ngroups = (int64_t(gridDim.x) * blockDim.x) / G;
    double acc = 0.0;
    for (int64_t i0 = gid - lane / G; i0 < m; i0 += ngroups) {  // warp-uniform bound
        const int64_t i = i0 + lane / G;
        const bool valid = i < m;
        const int64_t s = valid ? rowptr[i] : 0, e = valid ? rowptr[i + 1] : 0;
        const T r = group_row_dot(val, col, s, e, x, gl, G);
        if (valid && gl == 0) {
            const double c = double(violation(r, lb[i], ub[i]));
            const double delta = fabs(c) * invnorm[i];  // Euclidean distance to C_i; 0 for empty rows (A-4, A-5)
            if (mode == 0) acc += w[i] * delta * delta;
            else if (mode == 1) acc += w[i] * pow(delta, p);
            else acc = fmax(acc, delta);
        }
    }
    // block combine (sum or max), fixed order
    for (int o = 16; o > 0; o >>= 1) {
        double t = __shfl_xor_sync(0xffffffffu, acc, o);
        acc = mode == 2 ? fmax(acc, t) : acc + t;
    }
    if (lane == 0) ws[wid] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = ws[0];
        for (int q = 1; q < SUP_THREADS / 32; ++q) t = mode == 2 ? fmax(t, ws[q]) : t + ws[q];
        partials[blockIdx.x] = t;
    }
}

__global__ void k_prox_final(const double* __restrict__ partials, int np, int mode, double* __restrict__ out) {
    __shared__ double sh[SUP_THREADS];
    double s = 0.0;
    for (int q = threadIdx.x; q < np; q += SUP_THREADS) s = mode == 2 ? fmax(s, partials[q]) : s + partials[q];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = SUP_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] = mode == 2 ? fmax(sh[threadIdx.x], sh[threadIdx.x + o]) : sh[threadIdx.x] + sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = mode == 0 ? 0.5 * sh[0] : sh[0];
}

void sup_launch_proximity(sup_ctx* h, const void* x, int mode, double p, double* out_dev) {
    const int G = h->g_fwd;
    int cap = h->num_sms * 8;
    if (cap > SUP_MAX_PARTIALS) cap = SUP_MAX_PARTIALS;
    const int grid = sup_grid_for(h->m * G, SUP_THREADS, cap);
    if (h->dt == SUP_F32)
        k_prox<float><<<grid, SUP_THREADS, 0, h->stream>>>(
            h->m, h->A.rowptr, h->A.col, static_cast<const float*>(h->A.val), static_cast<const float*>(x),
            static_cast<const float*>(h->lb), static_cast<const float*>(h->ub), h->w, h->invnorm, mode, p, h->partials, G);
    else
        k_prox<double><<<grid, SUP_THREADS, 0, h->stream>>>(
            h->m, h->A.rowptr, h->A.col, static_cast<const double*>(h->A.val), static_cast<const double*>(x),
            static_cast<const double*>(h->lb), static_cast<const double*>(h->ub), h->w, h->invnorm, mode, p, h->partials, G);
    k_prox_final<<<1, SUP_THREADS, 0, h->stream>>>(h->partials, grid, mode, out_dev);
    h->launches += 2;
}
