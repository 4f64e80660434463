// sup_setup.cu -- S0 of the hot path: row norms, weights, d_i = w_i/||a_i||^2,
// input validation, and the explicit transposed CSR built by a stable LSD radix sort on the column index
// (stable => every row of A^T is sorted by original row index => the back-projection sums in a fixed order).
#include <math.h>
#include <stdarg.h>

#include "sup_internal.cuh"

char g_create_error[512] = {0};

sup_status sup_fail(sup_ctx* h, sup_status s, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(h ? h->err : g_create_error, 512, fmt, ap);
    va_end(ap);
    return s;
}

// ------------------------------------------------------------------------------------------------------------
// exclusive scan of a uint32 array (three-phase, recursive on the tile sums)
// ------------------------------------------------------------------------------------------------------------
#define SCAN_ITEMS 8
#define SCAN_TILE (SUP_THREADS * SCAN_ITEMS)

__device__ __forceinline__ unsigned block_exclusive_scan(unsigned v, unsigned* total) {
    __shared__ unsigned warp_sums[SUP_THREADS / 32];
    __shared__ unsigned block_total;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        unsigned s = lane < SUP_THREADS / 32 ? warp_sums[lane] : 0u;
        unsigned si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        if (lane < SUP_THREADS / 32) warp_sums[lane] = si - s;
        if (lane == 31) block_total = si;
    }
    __syncthreads();
    unsigned r = inc - v + warp_sums[wid];
    if (total) *total = block_total;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SUP_THREADS) k_scan_tile_sums(const unsigned* __restrict__ data, int64_t L,
                                                                unsigned* __restrict__ sums) {
    int64_t base = int64_t(blockIdx.x) * SCAN_TILE + int64_t(threadIdx.x) * SCAN_ITEMS;
    unsigned s = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q)
        if (base + q < L) s += data[base + q];
    unsigned total;
    block_exclusive_scan(s, &total);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(SUP_THREADS) k_scan_tile_apply(unsigned* __restrict__ data, int64_t L,
                                                                 const unsigned* __restrict__ sums) {
    int64_t base = int64_t(blockIdx.x) * SCAN_TILE + int64_t(threadIdx.x) * SCAN_ITEMS;
    unsigned v[SCAN_ITEMS];
    unsigned s = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q) {
        v[q] = base + q < L ? data[base + q] : 0u;
        s += v[q];
    }
    unsigned off = block_exclusive_scan(s, nullptr) + (sums ? sums[blockIdx.x] : 0u);
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q) {
        if (base + q < L) data[base + q] = off;
        off += v[q];
    }
}

static size_t scan_scratch_bytes(int64_t L) {
    size_t tot = 0;
    while (L > SCAN_TILE) {
        L = (L + SCAN_TILE - 1) / SCAN_TILE;
        tot += ((size_t(L) * 4 + 255) & ~size_t(255));
    }
    return tot + 256;
}

static void scan_exclusive_u32(sup_ctx* h, unsigned* data, int64_t L, char* scratch) {
    int64_t nb = (L + SCAN_TILE - 1) / SCAN_TILE;
    if (nb <= 1) {
        k_scan_tile_apply<<<1, SUP_THREADS, 0, h->stream>>>(data, L, nullptr);
        h->launches++;
        return;
    }
    unsigned* sums = reinterpret_cast<unsigned*>(scratch);
    k_scan_tile_sums<<<unsigned(nb), SUP_THREADS, 0, h->stream>>>(data, L, sums);
    h->launches++;
    scan_exclusive_u32(h, sums, nb, scratch + ((size_t(nb) * 4 + 255) & ~size_t(255)));
    k_scan_tile_apply<<<unsigned(nb), SUP_THREADS, 0, h->stream>>>(data, L, sums);
    h->launches++;
}

// ------------------------------------------------------------------------------------------------------------
// stable LSD radix sort pass (8-bit digits); one warp owns a chunk of RS_CHUNK consecutive items
// ------------------------------------------------------------------------------------------------------------
#define RS_ROUNDS 128
#define RS_CHUNK (32 * RS_ROUNDS)
#define RS_WARPS (SUP_THREADS / 32)

__global__ void __launch_bounds__(SUP_THREADS) k_radix_hist(const unsigned* __restrict__ keys, int64_t N, int shift,
                                                            unsigned* __restrict__ hist, int64_t nchunks) {
    __shared__ unsigned cnt[RS_WARPS][256];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t chunk = int64_t(blockIdx.x) * RS_WARPS + wid;
    for (int d = lane; d < 256; d += 32) cnt[wid][d] = 0;
    __syncwarp();
    if (chunk < nchunks) {
        const int64_t base = chunk * RS_CHUNK;
        for (int r = 0; r < RS_ROUNDS; ++r) {
            int64_t idx = base + int64_t(r) * 32 + lane;
            if (idx < N) atomicAdd(&cnt[wid][(keys[idx] >> shift) & 255u], 1u);
        }
        __syncwarp();
        for (int d = lane; d < 256; d += 32) hist[int64_t(d) * nchunks + chunk] = cnt[wid][d];
    }
}

template <typename T>
__global__ void __launch_bounds__(SUP_THREADS)
    k_radix_scatter(const unsigned* __restrict__ keys, const int* __restrict__ rows, const T* __restrict__ vals,
                    int64_t N, int shift, const unsigned* __restrict__ hist, int64_t nchunks,
                    unsigned* __restrict__ keys_out, int* __restrict__ rows_out, T* __restrict__ vals_out) {
    __shared__ unsigned off[RS_WARPS][256];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t chunk = int64_t(blockIdx.x) * RS_WARPS + wid;
    if (chunk >= nchunks) return;
    for (int d = lane; d < 256; d += 32) off[wid][d] = hist[int64_t(d) * nchunks + chunk];
    __syncwarp();
    const int64_t base = chunk * RS_CHUNK;
    const unsigned lt = (1u << lane) - 1u;
    for (int r = 0; r < RS_ROUNDS; ++r) {
        int64_t idx = base + int64_t(r) * 32 + lane;
        bool valid = idx < N;
        unsigned key = valid ? keys[idx] : 0u;
        unsigned dg = valid ? ((key >> shift) & 255u) : 256u;
        unsigned peers = __match_any_sync(0xffffffffu, dg);
        unsigned rank = __popc(peers & lt);
        unsigned pos = valid ? off[wid][dg] + rank : 0u;
        __syncwarp();
        if (valid && rank == 0) off[wid][dg] += __popc(peers);
        __syncwarp();
        if (valid) {
            keys_out[pos] = key;
            rows_out[pos] = rows[idx];
            vals_out[pos] = vals[idx];
        }
    }
}

// row index of every stored entry e in [e0, e0+N): the row i with rowptr[i] <= e < rowptr[i+1]
__global__ void __launch_bounds__(SUP_THREADS) k_expand_rows(const int64_t* __restrict__ rowptr, int64_t r0, int64_t r1,
                                                             int64_t e0, int64_t N, int* __restrict__ rows) {
    int64_t t = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (t >= N) return;
    int64_t e = e0 + t;
    int64_t lo = r0, hi = r1;  // invariant: rowptr[lo] <= e < rowptr[hi]
    while (hi - lo > 1) {
        int64_t mid = (lo + hi) >> 1;
        if (rowptr[mid] <= e) lo = mid; else hi = mid;
    }
    rows[t] = int(lo);
}

// rowptr of the transposed block from the sorted keys: out[j] = base + (number of keys < j)
__global__ void __launch_bounds__(SUP_THREADS) k_rowptr_from_keys(const unsigned* __restrict__ keys, int64_t N,
                                                                  int64_t cols, int64_t base,
                                                                  int64_t* __restrict__ out) {
    int64_t t = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
    if (t > N) return;
    int64_t prev = t == 0 ? -1 : int64_t(keys[t - 1]);
    int64_t cur = t == N ? cols : int64_t(keys[t]);
    for (int64_t j = prev + 1; j <= cur; ++j) out[j] = base + t;
}

size_t sup_transpose_scratch_bytes(int64_t N, int64_t cols, size_t esz) {
    (void)cols;
    size_t a4 = (size_t(N) * 4 + 255) & ~size_t(255);
    size_t av = (size_t(N) * esz + 255) & ~size_t(255);
    int64_t nchunks = (N + RS_CHUNK - 1) / RS_CHUNK;
    size_t hist = (size_t(nchunks) * 256 * 4 + 255) & ~size_t(255);
    return 4 * a4 + 2 * av + hist + scan_scratch_bytes(nchunks * 256) + 1024;
}

sup_status sup_transpose_rows(sup_ctx* h, const CsrD& A, int64_t r0, int64_t r1, int64_t e0, int64_t e1,
                              int64_t* out_rowptr, int32_t* out_col, void* out_val, int64_t out_base, void* scratch,
                              size_t scratch_bytes) {
    const int64_t N = e1 - e0;
    if (N > 0xfffffffeLL) return sup_fail(h, SUP_ERR_INVALID_ARG, "transpose: more than 2^32-2 entries in one block (32-bit unsigned ranks)");
    if (scratch_bytes < sup_transpose_scratch_bytes(N, A.cols, h->esz))
        return sup_fail(h, SUP_ERR_WORKSPACE, "transpose: scratch too small");
    cudaStream_t st = h->stream;
    if (N == 0) {
        k_rowptr_from_keys<<<1, SUP_THREADS, 0, st>>>(nullptr, 0, A.cols, out_base, out_rowptr);
        h->launches++;
        return SUP_OK;
    }
    Bump B{static_cast<char*>(scratch), scratch_bytes, 0, true};
    unsigned* key[2] = {static_cast<unsigned*>(B.take(size_t(N) * 4)), static_cast<unsigned*>(B.take(size_t(N) * 4))};
    int* row[2] = {static_cast<int*>(B.take(size_t(N) * 4)), static_cast<int*>(B.take(size_t(N) * 4))};
    void* val[2] = {B.take(size_t(N) * h->esz), B.take(size_t(N) * h->esz)};
    const int64_t nchunks = (N + RS_CHUNK - 1) / RS_CHUNK;
    unsigned* hist = static_cast<unsigned*>(B.take(size_t(nchunks) * 256 * 4));
    char* scan_scr = static_cast<char*>(B.take(scan_scratch_bytes(nchunks * 256)));
    if (!B.ok) return sup_fail(h, SUP_ERR_WORKSPACE, "transpose: scratch too small");

    int bits = 1;
    while ((int64_t(1) << bits) < A.cols) ++bits;
    const int passes = (bits + 7) / 8;

    k_expand_rows<<<unsigned((N + SUP_THREADS - 1) / SUP_THREADS), SUP_THREADS, 0, st>>>(A.rowptr, r0, r1, e0, N, row[0]);
    h->launches++;
    const unsigned* kin = reinterpret_cast<const unsigned*>(A.col + e0);
    const int* rin = row[0];
    const char* vin = static_cast<const char*>(A.val) + size_t(e0) * h->esz;
    const unsigned nb = unsigned((nchunks + RS_WARPS - 1) / RS_WARPS);
    for (int p = 0; p < passes; ++p) {
        const bool last = p == passes - 1;
        unsigned* kout = key[p & 1];
        int* rout = last ? out_col + (out_base) : row[(p + 1) & 1];
        char* vout = last ? static_cast<char*>(out_val) + size_t(out_base) * h->esz : static_cast<char*>(val[p & 1]);
        k_radix_hist<<<nb, SUP_THREADS, 0, st>>>(kin, N, 8 * p, hist, nchunks);
        h->launches++;
        scan_exclusive_u32(h, hist, nchunks * 256, scan_scr);
        if (h->dt == SUP_F32)
            k_radix_scatter<float><<<nb, SUP_THREADS, 0, st>>>(kin, rin, reinterpret_cast<const float*>(vin), N, 8 * p,
                                                               hist, nchunks, kout, rout, reinterpret_cast<float*>(vout));
        else
            k_radix_scatter<double><<<nb, SUP_THREADS, 0, st>>>(kin, rin, reinterpret_cast<const double*>(vin), N, 8 * p,
                                                                hist, nchunks, kout, rout, reinterpret_cast<double*>(vout));
        h->launches++;
        kin = kout;
        rin = rout;
        vin = vout;
    }
    k_rowptr_from_keys<<<unsigned((N + 1 + SUP_THREADS - 1) / SUP_THREADS), SUP_THREADS, 0, st>>>(kin, N, A.cols,
                                                                                                 out_base, out_rowptr);
    h->launches++;
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

// ------------------------------------------------------------------------------------------------------------
// weights, row norms, scaling, validation
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double ws[SUP_THREADS / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) ws[wid] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int q = 0; q < SUP_THREADS / 32; ++q) t += ws[q];
    return t;  // valid on thread 0
}

// flags: bit0 weight <= 0 or non-finite, bit1 lb > ub (or NaN), bit2 lo > hi (or NaN), bit3 column out of range,
//        bit4 columns not strictly increasing, bit5 rowptr not monotone / ends wrong
template <typename T>
__global__ void __launch_bounds__(SUP_THREADS) k_weight_sum(const T* __restrict__ w, int64_t m, double* __restrict__ partials,
                                                            int* __restrict__ flags) {
    double s = 0.0;
    int bad = 0;
    for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < m; i += int64_t(gridDim.x) * blockDim.x) {
        double wi = double(w[i]);
        if (!(wi > 0.0) || isinf(wi)) bad = 1;
        s += wi;
    }
    if (bad) atomicOr(flags, 1);
    s = block_sum(s);
    if (threadIdx.x == 0) partials[blockIdx.x] = s;
}

__global__ void k_sum_partials(const double* __restrict__ partials, int np, double* __restrict__ out) {
    __shared__ double sh[SUP_THREADS];
    double s = 0.0;
    for (int q = threadIdx.x; q < np; q += SUP_THREADS) s += partials[q];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = SUP_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

// one group of G lanes per row: rho_i = sum a_ij^2 (fp64), w_i, d_i, 1/||a_i||, structural checks
template <typename T>
__global__ void __launch_bounds__(SUP_THREADS)
    k_row_setup(int64_t m, int64_t n, int64_t nnz, const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
                const T* __restrict__ val, const T* __restrict__ w_in, const double* __restrict__ wsum,
                const T* __restrict__ lb, const T* __restrict__ ub, int G, T* __restrict__ d, double* __restrict__ w,
                double* __restrict__ invnorm, int* __restrict__ flags) {
    const int gl = threadIdx.x % G;
    const int lane = threadIdx.x & 31;
    const int64_t gid = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) / G;
    const int64_t ngroups = (int64_t(gridDim.x) * blockDim.x) / G;
    int bad = 0;
    // the loop bound is warp-uniform (first group of the warp) so that the shuffles below are never divergent
    for (int64_t i0 = gid - lane / G; i0 < m; i0 += ngroups) {
        const int64_t i = i0 + lane / G;
        const bool valid = i < m;
        int64_t s = valid ? rowptr[i] : 0, e = valid ? rowptr[i + 1] : 0;
        if (valid && (s > e || s < 0 || e > nnz || (i == 0 && s != 0) || (i == m - 1 && e != nnz))) {
            bad |= 32;
            s = e = 0;
        }
        double rho = 0.0;
        for (int64_t k = s + gl; k < e; k += G) {
            double v = double(val[k]);
            rho += v * v;
            int c = col[k];
            if (c < 0 || c >= n) bad |= 8;
            if (k > s && col[k - 1] >= c) bad |= 16;
        }
        for (int o = G >> 1; o > 0; o >>= 1) rho += __shfl_xor_sync(0xffffffffu, rho, o, G);
        if (valid && gl == 0) {
            double wi = w_in ? double(w_in[i]) / *wsum : 1.0 / double(m);
            w[i] = wi;
            d[i] = rho > 0.0 ? T(wi / rho) : T(0);
            invnorm[i] = rho > 0.0 ? 1.0 / sqrt(rho) : 0.0;
            if (!(lb[i] <= ub[i])) bad |= 2;
        }
    }
    if (bad) atomicOr(flags, bad);
}

template <typename T>
__global__ void __launch_bounds__(SUP_THREADS) k_check_box(const T* __restrict__ lo, const T* __restrict__ hi, int64_t n,
                                                           int* __restrict__ flags) {
    int bad = 0;
    for (int64_t j = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; j < n; j += int64_t(gridDim.x) * blockDim.x)
        if (!(lo[j] <= hi[j])) bad = 4;
    if (bad) atomicOr(flags, bad);
}

// structural check of a second matrix (dose): columns in range and increasing, rowptr monotone
__global__ void __launch_bounds__(SUP_THREADS) k_check_csr(int64_t m, int64_t n, int64_t nnz, const int64_t* __restrict__ rowptr,
                                                           const int32_t* __restrict__ col, int* __restrict__ flags) {
    int bad = 0;
    for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < m; i += int64_t(gridDim.x) * blockDim.x) {
        const int64_t s = rowptr[i], e = rowptr[i + 1];
        if (s > e || s < 0 || e > nnz || (i == 0 && s != 0) || (i == m - 1 && e != nnz)) {
            bad |= 32;
            continue;
        }
        for (int64_t k = s; k < e; ++k) {
            int c = col[k];
            if (c < 0 || c >= n) bad |= 8;
            if (k > s && col[k - 1] >= c) bad |= 16;
        }
    }
    if (bad) atomicOr(flags, bad);
}

// block-iterative scaling (A-14): d_blk_i = (w_i / W_t) / ||a_i||^2 = d_i / W_t, W_t = sum of w over block t
__global__ void __launch_bounds__(SUP_THREADS) k_block_weight(const double* __restrict__ w, int64_t r0, int64_t r1,
                                                              double* __restrict__ out) {
    // single CTA, fixed order: deterministic
    double s = 0.0;
    for (int64_t i = r0 + threadIdx.x; i < r1; i += SUP_THREADS) s += w[i];
    s = block_sum(s);
    if (threadIdx.x == 0) *out = s;
}
template <typename T>
__global__ void __launch_bounds__(SUP_THREADS) k_block_scale(const double* __restrict__ w, const double* __restrict__ invnorm,
                                                             int64_t r0, int64_t r1, const double* __restrict__ Wt,
                                                             T* __restrict__ d_blk) {
    for (int64_t i = r0 + int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < r1; i += int64_t(gridDim.x) * blockDim.x) {
        double inv = invnorm[i];
        d_blk[i] = (*Wt > 0.0) ? T((w[i] / *Wt) * inv * inv) : T(0);
    }
}

static sup_status flags_to_status(sup_ctx* h, int flags) {
    if (!flags) return SUP_OK;
    return sup_fail(h, SUP_ERR_FORMAT, "invalid input:%s%s%s%s%s%s", (flags & 1) ? " weight<=0" : "",
                    (flags & 2) ? " lb>ub" : "", (flags & 4) ? " box_lo>box_hi" : "", (flags & 8) ? " column out of range" : "",
                    (flags & 16) ? " columns not strictly increasing" : "", (flags & 32) ? " bad rowptr" : "");
}

sup_status sup_setup_rows(sup_ctx* h, const void* weights, void* scratch, size_t scratch_bytes) {
    if (scratch_bytes < 1024) return sup_fail(h, SUP_ERR_WORKSPACE, "setup: scratch too small");
    cudaStream_t st = h->stream;
    int* flags = static_cast<int*>(scratch);
    double* wsum = reinterpret_cast<double*>(static_cast<char*>(scratch) + 256);
    SUP_CUDA(h, cudaMemsetAsync(scratch, 0, 512, st));
    const int cap = h->num_sms * 8 < SUP_MAX_PARTIALS ? h->num_sms * 8 : SUP_MAX_PARTIALS;
    const int G = h->g_fwd;
    const int grid_rows = sup_grid_for(h->m * G, SUP_THREADS, h->num_sms * 16);
    if (h->dt == SUP_F32) {
        if (weights) {
            int gw = sup_grid_for(h->m, SUP_THREADS, cap);
            k_weight_sum<float><<<gw, SUP_THREADS, 0, st>>>(static_cast<const float*>(weights), h->m, h->partials, flags);
            k_sum_partials<<<1, SUP_THREADS, 0, st>>>(h->partials, gw, wsum);
            h->launches += 2;
        }
        k_row_setup<float><<<grid_rows, SUP_THREADS, 0, st>>>(
            h->m, h->n, h->nnz, h->A.rowptr, h->A.col, static_cast<const float*>(h->A.val),
            static_cast<const float*>(weights), wsum, static_cast<const float*>(h->lb), static_cast<const float*>(h->ub), G,
            static_cast<float*>(h->d), h->w, h->invnorm, flags);
        k_check_box<float><<<sup_grid_for(h->n, SUP_THREADS, cap), SUP_THREADS, 0, st>>>(
            static_cast<const float*>(h->lo), static_cast<const float*>(h->hi), h->n, flags);
    } else {
        if (weights) {
            int gw = sup_grid_for(h->m, SUP_THREADS, cap);
            k_weight_sum<double><<<gw, SUP_THREADS, 0, st>>>(static_cast<const double*>(weights), h->m, h->partials, flags);
            k_sum_partials<<<1, SUP_THREADS, 0, st>>>(h->partials, gw, wsum);
            h->launches += 2;
        }
        k_row_setup<double><<<grid_rows, SUP_THREADS, 0, st>>>(
            h->m, h->n, h->nnz, h->A.rowptr, h->A.col, static_cast<const double*>(h->A.val),
            static_cast<const double*>(weights), wsum, static_cast<const double*>(h->lb), static_cast<const double*>(h->ub),
            G, static_cast<double*>(h->d), h->w, h->invnorm, flags);
        k_check_box<double><<<sup_grid_for(h->n, SUP_THREADS, cap), SUP_THREADS, 0, st>>>(
            static_cast<const double*>(h->lo), static_cast<const double*>(h->hi), h->n, flags);
    }
    h->launches += 2;
    int hflags = 0;
    SUP_CUDA(h, cudaMemcpyAsync(&hflags, flags, sizeof(int), cudaMemcpyDeviceToHost, st));
    SUP_CUDA(h, cudaStreamSynchronize(st));
    return flags_to_status(h, hflags);
}

sup_status sup_validate(sup_ctx* h, const CsrD& M, bool check_bounds, void* scratch) {
    (void)check_bounds;
    cudaStream_t st = h->stream;
    int* flags = static_cast<int*>(scratch);
    SUP_CUDA(h, cudaMemsetAsync(scratch, 0, 256, st));
    k_check_csr<<<sup_grid_for(M.rows, SUP_THREADS, h->num_sms * 16), SUP_THREADS, 0, st>>>(M.rows, M.cols, M.nnz, M.rowptr,
                                                                                             M.col, flags);
    h->launches++;
    int hflags = 0;
    SUP_CUDA(h, cudaMemcpyAsync(&hflags, flags, sizeof(int), cudaMemcpyDeviceToHost, st));
    SUP_CUDA(h, cudaStreamSynchronize(st));
    return flags_to_status(h, hflags);
}

sup_status sup_setup_block_scaling(sup_ctx* h, void* scratch, size_t scratch_bytes) {
    if (scratch_bytes < size_t(h->n_blocks) * 8 + 256) return sup_fail(h, SUP_ERR_WORKSPACE, "blocks: scratch too small");
    double* Wt = static_cast<double*>(scratch);
    cudaStream_t st = h->stream;
    for (int t = 0; t < h->n_blocks; ++t) {
        const int64_t r0 = h->block_rowptr[t], r1 = h->block_rowptr[t + 1];
        k_block_weight<<<1, SUP_THREADS, 0, st>>>(h->w, r0, r1, Wt + t);
        const int grid = sup_grid_for(r1 - r0, SUP_THREADS, h->num_sms * 8);
        if (h->dt == SUP_F32)
            k_block_scale<float><<<grid, SUP_THREADS, 0, st>>>(h->w, h->invnorm, r0, r1, Wt + t, static_cast<float*>(h->d_blk));
        else
            k_block_scale<double><<<grid, SUP_THREADS, 0, st>>>(h->w, h->invnorm, r0, r1, Wt + t, static_cast<double*>(h->d_blk));
        h->launches += 2;
    }
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}
