// sup_static.cu -- sup_tv2d_value_static: the TV2D objective value (Eq. 15) with NO allocation and NO handle.
//
// Every other call of the library works on a handle whose workspace the caller allocated; the two-stage reductions keep their
// per-CTA partial sums there (k_objective + k_sum_final of sup_perturb.cu write h->partials).  Some callers cannot allocate at all
// at the point where they need a value -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc --
// so this ONE entry point keeps its scratch (one partial sum per image row and an arrival counter) in file-scope __device__ arrays
// of a fixed size: SUP_STATIC_MAX_ROWS rows, 128 KB, resident on every GPU that loads the library until the process exits.
//
// Host code must not hand the arrays' NAMES to a kernel (in host code the name is a host-side stand-in, not a device address):
// the device addresses are fetched with cudaGetSymbolAddress once per device, with that device current, and cached.
// The scratch is shared by every call on a device and keeps the last call's contents: the counter is cleared at the start of each
// call (and by the CTA that consumed it), every row slot a call reads was written by that call.  Calls that overlap on the GPU
// (two streams, two host threads) race on it -- the caller serialises them.
#include <mutex>

#include "sup_internal.cuh"

#define SUP_STATIC_THREADS 256
#define SUP_STATIC_MAX_DEVICES 64

static __device__ __align__(256) double g_static_rows[SUP_STATIC_MAX_ROWS];  // row i: sum over j of the TV terms (i, j)
static __device__ __align__(256) unsigned g_static_count[64];                 // [0]: CTAs that have stored their rows

// CTA sum in a fixed order: thread-strided partial sums, then a shared-memory tree
__device__ __forceinline__ double static_cta_sum(double v, double* sh) {
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int o = SUP_STATIC_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    const double r = sh[0];
    __syncthreads();
    return r;
}

// f(X) = sum_{i < ny-1, j < nx-1} sqrt((X[i+1][j] - X[i][j])^2 + (X[i][j+1] - X[i][j])^2), terms and sums in fp64.
// CTA b takes the rows b, b + grid, ...; the last CTA to arrive adds the row sums in row order and writes *out.
template <typename T>
__global__ void __launch_bounds__(SUP_STATIC_THREADS)
    k_tv2d_value_static(const T* __restrict__ X, int64_t ny, int64_t nx, double* __restrict__ rows, unsigned* __restrict__ count, double* __restrict__ out) {
    __shared__ double sh[SUP_STATIC_THREADS];
    __shared__ bool last;
    for (int64_t i = blockIdx.x; i < ny; i += gridDim.x) {
        double acc = 0.0;
        if (i + 1 < ny) {
            const T* r0 = X + i * nx;
            const T* r1 = r0 + nx;
            for (int64_t j = threadIdx.x; j + 1 < nx; j += SUP_STATIC_THREADS) {
                const double c = double(r0[j]);
                const double dx = double(r1[j]) - c, dy = double(r0[j + 1]) - c;
                acc += sqrt(fma(dx, dx, dy * dy));
            }
        }
        const double s = static_cta_sum(acc, sh);
        if (threadIdx.x == 0) rows[i] = s;
    }
    if (threadIdx.x == 0) {
        __threadfence();  // this CTA's row sums are visible before its arrival is
        last = atomicAdd(count, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double acc = 0.0;
    for (int64_t i = threadIdx.x; i < ny; i += SUP_STATIC_THREADS) acc += __ldcg(rows + i);
    const double f = static_cta_sum(acc, sh);
    if (threadIdx.x == 0) {
        *out = f;
        *count = 0;  // left clean for the next call (which clears it anyway)
    }
}

// device addresses of the two arrays, per device, fetched once with that device current
static std::mutex g_static_mutex;
static double* g_rows_ptr[SUP_STATIC_MAX_DEVICES];
static unsigned* g_count_ptr[SUP_STATIC_MAX_DEVICES];
static int g_static_sms[SUP_STATIC_MAX_DEVICES];

extern "C" sup_status sup_tv2d_value_static(const void* x, int dtype, int64_t ny, int64_t nx, double* out_dev, void* stream) {
    if (!x || !out_dev) return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_tv2d_value_static: NULL x or out_dev");
    if (dtype != SUP_F32 && dtype != SUP_F64) return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_tv2d_value_static: dtype must be SUP_F32 or SUP_F64");
    if (ny < 1 || nx < 1) return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_tv2d_value_static: ny and nx must be >= 1");
    if (ny > SUP_STATIC_MAX_ROWS || nx > (int64_t(1) << 31))
        return sup_fail(nullptr, SUP_ERR_INVALID_ARG,
                        "sup_tv2d_value_static: %lld x %lld is beyond the static scratch (at most %d rows of at most 2^31 pixels); use sup_objective on a handle",
                        (long long)ny, (long long)nx, SUP_STATIC_MAX_ROWS);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= SUP_STATIC_MAX_DEVICES)
        return sup_fail(nullptr, SUP_ERR_CUDA, "sup_tv2d_value_static: no current CUDA device (or its ordinal is >= %d)", SUP_STATIC_MAX_DEVICES);
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, x) != cudaSuccess || (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) ||
        (pa.type == cudaMemoryTypeDevice && pa.device != dev)) {
        cudaGetLastError();
        return sup_fail(nullptr, SUP_ERR_INVALID_ARG, "sup_tv2d_value_static: x must be device memory of the CURRENT device (%d)", dev);
    }
    double* rows = nullptr;
    unsigned* count = nullptr;
    int sms = 0;
    {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_rows_ptr[dev]) {  // set-up, once per device, with that device current
            void *pr = nullptr, *pc = nullptr;
            cudaError_t e = cudaGetSymbolAddress(&pr, g_static_rows);
            if (e == cudaSuccess) e = cudaGetSymbolAddress(&pc, g_static_count);
            int n_sm = 0;
            if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess || !pr || !pc || n_sm < 1) {
                cudaGetLastError();
                return sup_fail(nullptr, SUP_ERR_CUDA, "sup_tv2d_value_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
            }
            g_count_ptr[dev] = static_cast<unsigned*>(pc);
            g_static_sms[dev] = n_sm;
            g_rows_ptr[dev] = static_cast<double*>(pr);
        }
        rows = g_rows_ptr[dev];
        count = g_count_ptr[dev];
        sms = g_static_sms[dev];
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // the counter must start at zero whatever an earlier (possibly aborted) call left there
    cudaError_t e = cudaMemsetAsync(count, 0, sizeof(unsigned), st);
    if (e != cudaSuccess) return sup_fail(nullptr, SUP_ERR_CUDA, "sup_tv2d_value_static: cudaMemsetAsync: %s", cudaGetErrorString(e));
    const int64_t cap = int64_t(sms) * 8;
    const unsigned grid = unsigned(ny < cap ? ny : cap);
    if (dtype == SUP_F32) k_tv2d_value_static<float><<<grid, SUP_STATIC_THREADS, 0, st>>>(static_cast<const float*>(x), ny, nx, rows, count, out_dev);
    else k_tv2d_value_static<double><<<grid, SUP_STATIC_THREADS, 0, st>>>(static_cast<const double*>(x), ny, nx, rows, count, out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return sup_fail(nullptr, SUP_ERR_CUDA, "sup_tv2d_value_static: launch: %s", cudaGetErrorString(e));
    return SUP_OK;
}
