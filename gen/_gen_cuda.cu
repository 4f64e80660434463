// gen/_gen_cuda.cu -- device-side generator of BASELINE.json configs[4] (the throughput sweep): the same pure-integer counter
// hash as gen/workloads.py (hash3 / random_csr / config5_sweep_point), so the large points (up to ~4e9 stored entries) never
// exist on the host.  INPUT GENERATION ONLY -- none of the method's arithmetic.  Bit-identical to the NumPy recipe
// (tests/test_gpu_algorithms.py::test_device_generator_is_bit_identical).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

__host__ __device__ static inline uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__host__ __device__ static inline uint64_t hash3(uint64_t seed, uint64_t i, uint64_t t) {
    return mix64(mix64(seed ^ (i * 0x9E3779B97F4A7C15ULL)) + t * 0xD1B54A32D192ED03ULL);
}

// row i: k sorted distinct columns, one per stratum of width n/k; value ((h >> 40) + 1) / 2^24
__global__ void k_fill(int64_t m, int k, uint64_t seed, int32_t* __restrict__ col, float* __restrict__ val, int64_t* __restrict__ rowptr) {
    const int64_t total = m * int64_t(k);
    const uint64_t w = uint64_t(m / 2) / uint64_t(k);
    for (int64_t e = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; e < total; e += int64_t(gridDim.x) * blockDim.x) {
        const uint64_t i = uint64_t(e / k), t = uint64_t(e % k);
        const uint64_t h = hash3(seed, i, t);
        col[e] = int32_t(t * w + h % w);
        val[e] = float(double((h >> 40) + 1) / 16777216.0);
    }
    for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i <= m; i += int64_t(gridDim.x) * blockDim.x) rowptr[i] = i * k;
}

// u(tag, i) = ((hash3(seed + tag, i, 0) >> 40) + 1) / 2^24
__global__ void k_uniform(int64_t cnt, uint64_t seed, float* __restrict__ out32, double* __restrict__ out64) {
    for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < cnt; i += int64_t(gridDim.x) * blockDim.x) {
        const double u = double((hash3(seed, uint64_t(i), 0) >> 40) + 1) / 16777216.0;
        if (out32) out32[i] = float(u);
        if (out64) out64[i] = u;
    }
}

// bounds: ax_i = sum_t val * x*[col] in fp64, left to right, no contraction (what scipy's CSR mat-vec does on the host);
// delta_i = max(0.1 u(seed+2, i), 1e-3); lb = nextafter(round_down_f32(ax - delta), -inf), ub = nextafter(round_up_f32(ax + delta), +inf)
__global__ void k_bounds(int64_t m, int k, uint64_t seed, const int32_t* __restrict__ col, const float* __restrict__ val,
                         const float* __restrict__ xstar, float* __restrict__ lb, float* __restrict__ ub) {
    for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < m; i += int64_t(gridDim.x) * blockDim.x) {
        double ax = 0.0;
        for (int t = 0; t < k; ++t) ax = __dadd_rn(ax, __dmul_rn(double(val[i * k + t]), double(xstar[col[i * k + t]])));
        const double u = double((hash3(seed + 2, uint64_t(i), 0) >> 40) + 1) / 16777216.0;
        const double delta = fmax(__dmul_rn(0.1, u), 1e-3);
        lb[i] = nextafterf(__double2float_rd(__dsub_rn(ax, delta)), -INFINITY);
        ub[i] = nextafterf(__double2float_ru(__dadd_rn(ax, delta)), INFINITY);
    }
}

extern "C" int gen_cfg5_device(int64_t m, int k, uint64_t seed, int64_t* rowptr, int32_t* col, float* val, float* xstar, float* lb, float* ub,
                               void* stream) {
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    k_fill<<<148 * 16, 256, 0, st>>>(m, k, seed, col, val, rowptr);
    k_uniform<<<148 * 4, 256, 0, st>>>(m / 2, seed + 1, xstar, nullptr);
    k_bounds<<<148 * 8, 256, 0, st>>>(m, k, seed, col, val, xstar, lb, ub);
    return int(cudaGetLastError());
}
