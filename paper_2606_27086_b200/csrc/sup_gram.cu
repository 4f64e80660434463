// sup_gram.cu -- the dose objective f(x) = ||D x||^2 (A-15) through its Gram matrix G = D^T D.
//
// Radiotherapy dose matrices are tall: config 4 has m = 1.34 M voxel rows and n = 8 000 beamlet columns, 74 M stored entries.  The
// perturbation phase needs, per reduction step, g = 2 D^T D x and ||D g||^2 = g^T (D^T D) g -- two passes over D (0.6 GB each) on
// the product kernels.  G = D^T D is n x n DENSE (256 MB in fp32 at n = 8 000, less than half of one pass over D) and turns the
// whole phase into 1 + N dense matrix-vector products in n-space:
//     pass 0:   u = G x;   f(x) = x^T u,  g_0 = 2 u,  ||g_0||^2 = 4 u^T u
//     step n:   w = G g_n; ||D g_n||^2 = g_n^T w;  trial loop on the closed form f(x - c g) = f(x) - c ||g||^2 + c^2 ||D g||^2
//               (as in the matrix-pass sequence of sup_algos.cu);  x <- x - c g_n,  g_{n+1} = g_n - 2 c w,  f <- the closed form.
// G is built once in sup_set_dose_matrix, deterministically (no atomics: a fixed summation order per entry), with fp64 accumulators,
// and stored in the handle's type.  The path is taken when n <= 16 384 and n^2 <= 2 nnz(D) (then one product with G moves fewer
// bytes than one pass over D); otherwise, or after sup_set_dose_mode(h, 1), the matrix-pass sequence runs.
//
// Kernels: k_gram_build (setup), k_gram_matvec (HBM-bound dense product, one CTA per SM, the vector in shared memory, four rows in
// flight per thread), k_gram_trial (the scalar trial loop, one thread), k_gram_apply (the two n-vector updates).
#include "sup_internal.cuh"

bool sup_gram_applicable(int64_t n, int64_t nnz) { return n >= 1 && n <= 16384 && n * n <= 2 * nnz; }
int64_t sup_gram_ld(int64_t n) { return (n + 31) & ~int64_t(31); }

// ---- setup: row j of G = sum over the entries (i, d_ij) of column j of D, in increasing i, of d_ij * (row i of D) ------------------
// One CTA per column j, the row of G in shared memory as fp64.  Warp w owns the slice [c0, c1) of the row and walks ALL rows i of the
// column in order, adding only the entries that fall into its slice: no two warps touch the same accumulator, a warp's updates are
// in program order, so every entry of G is summed in one fixed order (increasing i).
#define GRAM_BUILD_THREADS 256
template <typename T>
__global__ void __launch_bounds__(GRAM_BUILD_THREADS)
    k_gram_build(int n, int64_t ld, const int64_t* __restrict__ dt_rowptr, const int32_t* __restrict__ dt_col, const T* __restrict__ dt_val,
                 const int64_t* __restrict__ d_rowptr, const int32_t* __restrict__ d_col, const T* __restrict__ d_val, T* __restrict__ G) {
    extern __shared__ double gram_acc[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = GRAM_BUILD_THREADS / 32;
    const int per = (n + nw - 1) / nw;
    const int c0 = min(n, warp * per), c1 = min(n, c0 + per);
    for (int64_t j = blockIdx.x; j < n; j += gridDim.x) {
        for (int q = c0 + lane; q < c1; q += 32) gram_acc[q] = 0.0;
        __syncwarp();
        const int64_t p0 = dt_rowptr[j], p1 = dt_rowptr[j + 1];
        for (int64_t pb = p0; pb < p1; pb += 32) {
            // 32 entries of the column at a time: lane l fetches row index, value and row extent of entry pb + l
            const int64_t p = pb + lane;
            int64_t e0 = 0, e1 = 0;
            double dij = 0.0;
            if (p < p1) {
                const int i = dt_col[p];
                dij = double(dt_val[p]);
                e0 = d_rowptr[i];
                e1 = d_rowptr[i + 1];
            }
            const int cnt = int(p1 - pb < 32 ? p1 - pb : 32);
            for (int k = 0; k < cnt; k += 2) {  // two rows per trip, their loads issued before either update
                const int k2 = min(k + 1, cnt - 1);
                const int64_t a0 = __shfl_sync(0xffffffffu, e0, k), a1 = __shfl_sync(0xffffffffu, e1, k);
                const int64_t b0 = __shfl_sync(0xffffffffu, e0, k2), b1 = k2 == k ? b0 : __shfl_sync(0xffffffffu, e1, k2);
                const double da = __shfl_sync(0xffffffffu, dij, k), db = __shfl_sync(0xffffffffu, dij, k2);
                int ca[2], cb[2];
                double va[2], vb[2];
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const int64_t ea = a0 + 32 * t + lane, eb = b0 + 32 * t + lane;
                    ca[t] = ea < a1 ? d_col[ea] : -1;
                    va[t] = ea < a1 ? double(d_val[ea]) : 0.0;
                    cb[t] = eb < b1 ? d_col[eb] : -1;
                    vb[t] = eb < b1 ? double(d_val[eb]) : 0.0;
                }
#pragma unroll
                for (int t = 0; t < 2; ++t)
                    if (ca[t] >= c0 && ca[t] < c1) gram_acc[ca[t]] = fma(da, va[t], gram_acc[ca[t]]);
                for (int64_t e = a0 + 64 + lane; e < a1; e += 32) {  // rows of more than 64 entries
                    const int c = d_col[e];
                    if (c >= c0 && c < c1) gram_acc[c] = fma(da, double(d_val[e]), gram_acc[c]);
                }
                __syncwarp();
                if (k2 != k) {
#pragma unroll
                    for (int t = 0; t < 2; ++t)
                        if (cb[t] >= c0 && cb[t] < c1) gram_acc[cb[t]] = fma(db, vb[t], gram_acc[cb[t]]);
                    for (int64_t e = b0 + 64 + lane; e < b1; e += 32) {
                        const int c = d_col[e];
                        if (c >= c0 && c < c1) gram_acc[c] = fma(db, double(d_val[e]), gram_acc[c]);
                    }
                    __syncwarp();
                }
            }
        }
        __syncwarp();
        for (int q = c0 + lane; q < c1; q += 32) G[j * ld + q] = T(gram_acc[q]);
        if (warp == nw - 1)
            for (int64_t q = n + lane; q < ld; q += 32) G[j * ld + q] = T(0);  // the padding of the row
        __syncwarp();
    }
}

// ---- y = scale * G v with the reductions sum v_j u_j and sum u_j^2 (u = G v) ----------------------------------------------------
// One CTA per SM, rows split evenly; the vector sits in shared memory; all warps of the CTA share each row (a row of n = 8 000 fp32
// is 32 KB: one 16-byte load per thread and trip), four rows in flight per thread.  Products and the per-thread partial sums in the
// handle's type (chains of ld / (16/sizeof(T) * threads) terms), everything after that in fp64, in a fixed order.
#define GRAM_MV_WARPS 32
#ifndef GRAM_MV_ROWS
#define GRAM_MV_ROWS 4
#endif
template <typename T>
struct GramVec;
template <>
struct GramVec<float> {
    typedef float4 V;
    static __device__ __forceinline__ float dot(const float4& a, const float4& b, float acc) {
        acc = fmaf(a.x, b.x, acc);
        acc = fmaf(a.y, b.y, acc);
        acc = fmaf(a.z, b.z, acc);
        return fmaf(a.w, b.w, acc);
    }
};
template <>
struct GramVec<double> {
    typedef double2 V;
    static __device__ __forceinline__ double dot(const double2& a, const double2& b, double acc) { return fma(a.y, b.y, fma(a.x, b.x, acc)); }
};

template <typename T, bool VG>
__global__ void __launch_bounds__(32 * GRAM_MV_WARPS, 1)
    k_gram_matvec(const T* __restrict__ G, int n, int64_t ld, const T* __restrict__ v, double scale, T* __restrict__ out,
                  double* __restrict__ red_vu, double* __restrict__ red_uu, const DevState* __restrict__ st) {
    if (*(volatile const int*)&st->stop) return;
    typedef typename GramVec<T>::V V;
    constexpr int VEC = 16 / int(sizeof(T));
    extern __shared__ __align__(16) unsigned char gram_smem[];
    T* vs = reinterpret_cast<T*>(gram_smem);                                                // [ld]
    double* part = reinterpret_cast<double*>(gram_smem + ((size_t(ld) * sizeof(T) + 15) & ~size_t(15)));  // [rows_per_cta][GRAM_MV_WARPS]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (!VG) {
        for (int64_t q = threadIdx.x; q < ld; q += blockDim.x) vs[q] = q < n ? v[q] : T(0);
        __syncthreads();
    }
    const int r0 = int(int64_t(blockIdx.x) * n / gridDim.x), r1 = int(int64_t(blockIdx.x + 1) * n / gridDim.x);  // rows split evenly (+-1)
    const int nvec = int(ld / VEC);
    // VG: v is 16-byte aligned and read through L1 (32 KB at n = 8 000: it stays there), which saves the staging pass and its barrier;
    // the last, partial vector of v is assembled from scalars (G's padding is zero, v's does not exist)
    const V* vsv = reinterpret_cast<const V*>(VG ? v : vs);
    const int nfull = n / VEC;
    for (int r = r0; r < r1; r += GRAM_MV_ROWS) {
        const V* gp[GRAM_MV_ROWS];
        T acc[GRAM_MV_ROWS];
#pragma unroll
        for (int u = 0; u < GRAM_MV_ROWS; ++u) {
            gp[u] = reinterpret_cast<const V*>(G + int64_t(min(r + u, r1 - 1)) * ld);  // rows past the end repeat the last one (discarded)
            acc[u] = T(0);
        }
        for (int c = threadIdx.x; c < nvec; c += blockDim.x) {
            V a[GRAM_MV_ROWS];
#pragma unroll
            for (int u = 0; u < GRAM_MV_ROWS; ++u) a[u] = __ldcs(gp[u] + c);
            V b;
            if (!VG) {
                b = vsv[c];
            } else if (c < nfull) {
                b = __ldg(vsv + c);
            } else {
                T t[VEC];
#pragma unroll
                for (int e = 0; e < VEC; ++e) t[e] = c * VEC + e < n ? __ldg(v + c * VEC + e) : T(0);
                b = *reinterpret_cast<const V*>(t);
            }
#pragma unroll
            for (int u = 0; u < GRAM_MV_ROWS; ++u) acc[u] = GramVec<T>::dot(a[u], b, acc[u]);
        }
#pragma unroll
        for (int u = 0; u < GRAM_MV_ROWS; ++u) {
            double s = double(acc[u]);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0 && r + u < r1) part[(r + u - r0) * GRAM_MV_WARPS + warp] = s;
        }
    }
    __syncthreads();
    // row sums in warp order, the outputs and this CTA's share of the two reductions
    __shared__ double s_vu[32 * GRAM_MV_WARPS / 32], s_uu[32 * GRAM_MV_WARPS / 32];
    double pvu = 0.0, puu = 0.0;
    for (int rl = threadIdx.x; rl < r1 - r0; rl += blockDim.x) {
        double u = 0.0;
        for (int w = 0; w < GRAM_MV_WARPS; ++w) u += part[rl * GRAM_MV_WARPS + w];
        out[r0 + rl] = T(scale * u);
        pvu += double(v[r0 + rl]) * u;
        puu += u * u;
    }
    // rows_per_cta <= blockDim.x: thread rl holds row rl's terms; sum them in row order
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        pvu += __shfl_xor_sync(0xffffffffu, pvu, o);
        puu += __shfl_xor_sync(0xffffffffu, puu, o);
    }
    if (lane == 0) {
        s_vu[warp] = pvu;
        s_uu[warp] = puu;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < GRAM_MV_WARPS; ++w) {
            a += s_vu[w];
            b += s_uu[w];
        }
        red_vu[blockIdx.x] = a;
        red_uu[blockIdx.x] = b;
    }
}

// ---- the scalar part of a reduction step (one warp for the sums, one thread for the rest) -----------------------------------------------------------------------------
// sum of np per-CTA partials by one warp: lane l adds entries l, l + 32, ..., then a butterfly -- a fixed order
__device__ __forceinline__ double gram_sum(const double* __restrict__ p, int np) {
    double s = 0.0;
    for (int q = threadIdx.x; q < np; q += 32) s += __ldcg(p + q);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    return s;
}
// first: f(x) = sum x u and ||g_0||^2 = 4 sum u^2 from pass 0; later steps: f carried as the closed form, ||g||^2 from k_gram_apply.
// q2 = g^T G g = ||D g||^2 of this step.  final_only: only closes the phase (st->f, the adaptive rule's reference).
__global__ void k_gram_trial(DevState* st, const double* __restrict__ red_xu, const double* __restrict__ red_uu, int np_mv,
                             const double* __restrict__ red_gw, const double* __restrict__ part_gg, int np_apply, int first, int final_only,
                             double beta0, double a, int policy, long long n_restart, int8_t* decisions, double* decision_f, long long cap,
                             int step_rule, double shrink) {
    if (st->stop) return;
    sup_pdl_trigger();
    const long long k = st->k;
    if (final_only) {
        if (threadIdx.x != 0) return;
        st->f = st->f_cur;
        if (step_rule == SUP_RULE_ADAPTIVE && st->f_start <= st->f_ref) st->f_ref = shrink * st->f_start;  // A-30
        return;
    }
    if (threadIdx.x == 0 && first && n_restart > 0 && k > 0 && k % n_restart == 0) {  // restarted perturbations (A-24)
        st->ell = k / n_restart;
        st->apow = 1.0;
        for (long long q = 0; q < st->ell; ++q) st->apow *= a;
    }
    double fx = st->f_cur, s2;
    if (first) {
        fx = gram_sum(red_xu, np_mv);
        s2 = 4.0 * gram_sum(red_uu, np_mv);
    } else {
        s2 = gram_sum(part_gg, np_apply);
    }
    const double q2 = gram_sum(red_gw, np_mv);
    if (threadIdx.x != 0) return;  // the warp did the sums; one thread runs the trial loop
    if (first) st->f_start = fx;
    if (!isfinite(fx)) atomicOr(&st->fault, 2);
    st->f_cur = fx;
    st->f = fx;
    st->cf = 0.0;
    const double s = sqrt(s2);
    if (step_rule == SUP_RULE_ADAPTIVE) {  // Eq. 11 (A-30): no trial loop
        const bool take = fx > st->f_ref && s > 0.0;
        if (take) {
            const double c = ((fx - st->f_ref) / s) / s;
            st->cf = c;
            st->f_cur = fx - c * s2 + c * c * q2;
            st->n_trials += 1;
            st->sweep_trials += 1;
        }
        if (decisions && st->n_dec < cap) decisions[st->n_dec] = take ? 1 : 0;
        if (decision_f && st->n_dec < cap) {
            decision_f[2 * st->n_dec] = st->f_ref;
            decision_f[2 * st->n_dec + 1] = fx;
        }
        st->n_dec += 1;
        return;
    }
    bool accepted = false;
    long long jloc = 0;
    for (int trial = 0; trial < SUP_J_MAX && !accepted; ++trial) {
        double ap = st->apow;
        if (policy != SUP_STEP_PER_TRIAL) {
            ap = 1.0;
            for (long long q = 0; q < k + jloc; ++q) ap *= a;
        }
        const double c = s > 0.0 ? (beta0 * ap) / s : 0.0;
        const double fz = c == 0.0 ? fx : fx - c * s2 + c * c * q2;
        st->ell += 1;
        st->apow *= a;
        ++jloc;
        st->n_trials += 1;
        st->sweep_trials += 1;
        const bool acc = fz <= fx;  // NaN compares false (A-11)
        if (decisions && st->n_dec < cap) decisions[st->n_dec] = acc ? 1 : 0;
        if (decision_f && st->n_dec < cap) {
            decision_f[2 * st->n_dec] = fz;
            decision_f[2 * st->n_dec + 1] = fx;
        }
        st->n_dec += 1;
        if (acc) {
            accepted = true;
            st->cf = c;
            st->f_cur = fz;
        }
    }
    if (!accepted) atomicOr(&st->warn, 1);  // A-12: step skipped
}

// x <- round_T(x - c g), g <- round_T(g - 2 c w) (the gradient at the new point), per-CTA sums of the new g^2; the gather mirror of x
// is refreshed by the last step of the phase
template <typename T>
__global__ void __launch_bounds__(SUP_THREADS)
    k_gram_apply(const DevState* __restrict__ st, T* __restrict__ x, T* __restrict__ g, const T* __restrict__ w, int64_t n, T* __restrict__ xg,
                 const GMap xmap, double* __restrict__ partials) {
    if (st->stop) return;
    __shared__ double ws[SUP_THREADS];
    const double cf = st->cf;
    double gg = 0.0;
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n; j += int64_t(gridDim.x) * blockDim.x) {
        T xv = x[j], gv = g[j];
        if (cf != 0.0) {
            xv = T(fma(-cf, double(gv), double(xv)));
            gv = T(fma(-2.0 * cf, double(w[j]), double(gv)));
            x[j] = xv;
            g[j] = gv;
        }
        if (xg) xg[sup_gmap(xmap, int(j))] = xv;
        gg += double(gv) * double(gv);
    }
    ws[threadIdx.x] = gg;
    __syncthreads();
    for (int o = SUP_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) ws[threadIdx.x] += ws[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = ws[0];
}

// ---- host side ----------------------------------------------------------------------------------------------------------------------
static int gram_mv_grid(const sup_ctx* h) { return int(std::min<int64_t>(h->n, h->num_sms)); }
static int gram_rows_per_cta(const sup_ctx* h) { return int((h->n + gram_mv_grid(h) - 1) / gram_mv_grid(h)); }
static size_t gram_mv_smem(const sup_ctx* h) {
    return ((size_t(h->gram_ld) * h->esz + 15) & ~size_t(15)) + size_t(gram_rows_per_cta(h)) * GRAM_MV_WARPS * sizeof(double);
}
template <typename T>
static sup_status gram_build_t(sup_ctx* h) {
    const int n = int(h->n);
    const size_t smem = size_t(n) * sizeof(double);
    // both kernels opt in to the device's maximum once (the attribute is per function, not per handle)
    int optin = 0;
    SUP_CUDA(h, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device));
    cudaFuncAttributes fb, fm;
    SUP_CUDA(h, cudaFuncGetAttributes(&fb, k_gram_build<T>));
    SUP_CUDA(h, cudaFuncGetAttributes(&fm, k_gram_matvec<T, false>));
    const int dyn_b = optin - int(fb.sharedSizeBytes), dyn_m = optin - int(fm.sharedSizeBytes);
    if (int64_t(smem) > dyn_b || int64_t(gram_mv_smem(h)) > dyn_m) return sup_fail(h, SUP_ERR_STATE, "Gram path: shared memory of this device is too small");
    SUP_CUDA(h, cudaFuncSetAttribute(k_gram_build<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_b));
    SUP_CUDA(h, cudaFuncSetAttribute(k_gram_matvec<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_m));
    SUP_CUDA(h, cudaFuncSetAttribute(k_gram_matvec<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_m));
    int per_sm = 1;
    SUP_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_gram_build<T>, GRAM_BUILD_THREADS, smem));
    const int grid = int(std::min<int64_t>(n, int64_t(h->num_sms) * std::max(per_sm, 1)));
    k_gram_build<T><<<grid, GRAM_BUILD_THREADS, smem, h->stream>>>(n, h->gram_ld, h->DT.rowptr, h->DT.col, static_cast<const T*>(h->DT.val), h->D.rowptr,
                                                                 h->D.col, static_cast<const T*>(h->D.val), static_cast<T*>(h->gram));
    h->launches++;
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}
sup_status sup_gram_build(sup_ctx* h) { return h->dt == SUP_F32 ? gram_build_t<float>(h) : gram_build_t<double>(h); }

template <typename T>
static sup_status gram_matvec_t(sup_ctx* h, const void* v, double scale, void* out, double* red_vu, double* red_uu) {
    const int grid = gram_mv_grid(h);
    const size_t smem = gram_mv_smem(h);
    if ((reinterpret_cast<uintptr_t>(v) & 15u) == 0)
        k_gram_matvec<T, true><<<grid, 32 * GRAM_MV_WARPS, smem, h->stream>>>(static_cast<const T*>(h->gram), int(h->n), h->gram_ld, static_cast<const T*>(v),
                                                                             scale, static_cast<T*>(out), red_vu, red_uu, h->state);
    else
        k_gram_matvec<T, false><<<grid, 32 * GRAM_MV_WARPS, smem, h->stream>>>(static_cast<const T*>(h->gram), int(h->n), h->gram_ld, static_cast<const T*>(v),
                                                                              scale, static_cast<T*>(out), red_vu, red_uu, h->state);
    h->launches++;
    return SUP_OK;
}

sup_status sup_launch_perturb_dose_gram(sup_ctx* h, void* x, const PerturbParams& pp) {
    double *red_xu = h->red, *red_uu = h->red + SUP_STREAM_NBMAX, *red_gw = h->red + 2 * SUP_STREAM_NBMAX;
    double* red_scratch = h->partials + SUP_MAX_PARTIALS;  // sum w^2 of the step products: not needed
    const int np_mv = gram_mv_grid(h);
    const int grid = sup_grid_for(h->n, SUP_THREADS, h->num_sms);
    void* mirror = pp.write_mirror && sup_stream_forward_uses_xg(h) ? h->xg : nullptr;
    const bool f32 = h->dt == SUP_F32;
    sup_status rc = f32 ? gram_matvec_t<float>(h, x, 2.0, h->g, red_xu, red_uu) : gram_matvec_t<double>(h, x, 2.0, h->g, red_xu, red_uu);  // g = 2 G x
    if (rc != SUP_OK) return rc;
    for (int nred = 0; nred < pp.N; ++nred) {
        rc = f32 ? gram_matvec_t<float>(h, h->g, 1.0, h->gram_w, red_gw, red_scratch) : gram_matvec_t<double>(h, h->g, 1.0, h->gram_w, red_gw, red_scratch);  // w = G g
        if (rc != SUP_OK) return rc;
        k_gram_trial<<<1, 32, 0, h->stream>>>(h->state, red_xu, red_uu, np_mv, red_gw, h->partials, grid, nred == 0, 0, pp.beta0, pp.a, pp.policy, pp.n_restart,
                                             pp.decisions, pp.decision_f, pp.cap, pp.step_rule, pp.shrink);
        void* mir = nred == pp.N - 1 ? mirror : nullptr;
        if (f32)
            k_gram_apply<float><<<grid, SUP_THREADS, 0, h->stream>>>(h->state, static_cast<float*>(x), static_cast<float*>(h->g), static_cast<const float*>(h->gram_w),
                                                                     h->n, static_cast<float*>(mir), h->xmap, h->partials);
        else
            k_gram_apply<double><<<grid, SUP_THREADS, 0, h->stream>>>(h->state, static_cast<double*>(x), static_cast<double*>(h->g),
                                                                      static_cast<const double*>(h->gram_w), h->n, static_cast<double*>(mir), h->xmap, h->partials);
        h->launches += 2;
    }
    k_gram_trial<<<1, 32, 0, h->stream>>>(h->state, red_xu, red_uu, np_mv, red_gw, h->partials, grid, 0, 1, pp.beta0, pp.a, pp.policy, pp.n_restart, pp.decisions,
                                         pp.decision_f, pp.cap, pp.step_rule, pp.shrink);
    h->launches++;
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}
