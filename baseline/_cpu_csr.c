/* baseline/_cpu_csr.c -- builder's CPU restatement of one simultaneous hyperslab sweep in plain fp64 with OpenMP (all host
 * cores): a REPORTED BASELINE for bench.py, not the oracle (oracle/) and not the product.  Forward product row-parallel over
 * A, back-projection row-parallel over an explicit transposed CSR, double accumulators.
 *   y_i = d_i c_i(<a_i, x>),  x_j <- clip(x_j - lambda sum_i a_ij y_i) */
#include <omp.h>
#include <stdint.h>

int cpu_threads(void) { return omp_get_max_threads(); }

void cpu_setup(int64_t m, const int64_t* rowptr, const double* val, double* d) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < m; ++i) {
        double rho = 0.0;
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) rho += val[k] * val[k];
        d[i] = rho > 0.0 ? (1.0 / (double)m) / rho : 0.0;
    }
}

void cpu_sweep(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const int64_t* trowptr,
               const int32_t* tcol, const double* tval, const double* lb, const double* ub, const double* d, const double* lo,
               const double* hi, double lambda, double* x, double* y) {
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < m; ++i) {
        double r = 0.0;
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) r += val[k] * x[col[k]];
        const double c = r > ub[i] ? r - ub[i] : (r < lb[i] ? r - lb[i] : 0.0);
        y[i] = d[i] * c;
    }
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t j = 0; j < n; ++j) {
        double u = 0.0;
        for (int64_t k = trowptr[j]; k < trowptr[j + 1]; ++k) u += tval[k] * y[tcol[k]];
        double t = x[j] - lambda * u;
        if (t < lo[j]) t = lo[j];
        if (t > hi[j]) t = hi[j];
        x[j] = t;
    }
}
