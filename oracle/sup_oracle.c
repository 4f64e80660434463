/*
 * oracle/sup_oracle.c -- plain, slow, fp64 CPU ORACLE of the superiorized simultaneous-projection path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code with the CUDA path
 * (paper_2606_27086_b200/csrc) and is written from the paper alone:
 *   /root/reference/PAPER.md = arXiv 2606.27086 (SupPy), cited as PAPER.md:L<line>.
 * Scalar loops, CSR traversed in storage order, back-projection as a scatter (no transposed matrix).
 * Every value is an fp64 number and every elementwise operation is one IEEE-754 fp64 operation (built with
 * -ffp-contract=off: no fused multiply-add).  Every REDUCTION (row dot product, back-projected sum, ||a_i||^2,
 * weight sums, objective sums, ||g||^2) is accumulated in binary128 (acc_t) and rounded once to fp64: a product
 * of two fp64 numbers is exact in binary128, so the result is the correctly rounded fp64 value of the sum and
 * does not depend on summation order (reading A-22: the perturbed iteration amplifies last-bit
 * differences by orders of magnitude per sweep, so "the sum" has to be one well-defined number).
 * Readings of the paper where it is silent/garbled are listed in DESIGN.md ("Readings", A-1 .. A-30) and
 * named at the line that uses them.
 *
 * Parity pins (tests/test_oracle_pins.py): every function below is pinned by closed forms, invariants,
 * library special cases or brute force -- the hyperslab sweeps, proximities, TV2D/TV1D/dose objectives and Algorithm 1
 * (round 1), and DROP / EMR (dense NumPy expression of Table A.5, exact line minimiser), f_Mean (linearity, exact
 * decrease -beta ||g||), TV3D (closed forms, finite differences, reduction to TV2D) and the stopping rule (replay from
 * the definition; never firing = bit-identical fixed run), and Eq. 11's step (half-space projection: f lands on f_ref
 * exactly for a linear f, Heron's square-root iteration for f = x^2).  PARITY UNPINNED: the f_ref update rule inside
 * orc_perturb_adaptive (reading A-30) -- the paper only cites the rule, so no value of it can be checked against the paper.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef __float128 acc_t; /* accumulator of every reduction (A-22) */

typedef struct {
    int64_t m, n;
    const int64_t* rowptr;
    const int32_t* col;
    const double* val;
} csr_t;

/* ---- O-SETUP: weights and row scaling.  PAPER.md:L63 (w_i > 0, sum w_i = 1), L608 (D = diag(w_i/||a^i||^2)).
 * A-3: no weights => 1/m; given weights are divided by their sum.  A-4: empty rows get d_i = 0.
 * Returns 0, or 1 if a weight is not > 0. */
int orc_setup(int64_t m, const int64_t* rowptr, const int32_t* col, const double* val, const double* w_in,
              double* w, double* rho, double* d) {
    (void)col;
    acc_t sw_acc = 0;
    for (int64_t i = 0; i < m; ++i) {
        double wi = w_in ? w_in[i] : 1.0;
        if (!(wi > 0.0)) return 1;
        sw_acc += wi;
    }
    const double sw = (double)sw_acc;
    for (int64_t i = 0; i < m; ++i) {
        w[i] = (w_in ? w_in[i] : 1.0) / sw;
        acc_t r_acc = 0;
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) r_acc += (acc_t)val[k] * val[k]; /* ||a^i||^2 */
        const double r = (double)r_acc;
        rho[i] = r;
        d[i] = r > 0.0 ? w[i] / r : 0.0;
    }
    return 0;
}

/* hyperslab violation of row value r against [lb, ub]: Eq. 2 applied to each face of
 * lb <= <a,x> <= ub (Eq. 20); at most one face is violated. */
static double violation(double r, double lb, double ub) {
    if (r > ub) return r - ub;
    if (r < lb) return r - lb;
    return 0.0;
}

/* <a^i, x>: the products are exact in binary128, the sum is rounded once to fp64 (A-22) */
static double row_dot(const int64_t* rowptr, const int32_t* col, const double* val, int64_t i, const double* x) {
    acc_t r = 0;
    for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) r += (acc_t)val[k] * x[col[k]];
    return (double)r;
}

/* ---- O-SWEEP on rows [r0, r1): x <- P_box(x - lambda * A^T D c(x)).
 * A-1: T(x) = x + lambda * sum_i w_i (P_{C_i}(x) - x)  (Eq. 2, 3 and the weights of Eq. 5 / Table A.5's D).
 * A-2: the box is applied after the relaxed step, un-relaxed.
 * dscale multiplies d_i (1 for the simultaneous sweep; 1/W_t for block t, A-14).  u is scratch [n]. */
static void sweep_rows(const csr_t* A, int64_t r0, int64_t r1, const double* lb, const double* ub, const double* d,
                       double dscale, const double* lo, const double* hi, double lambda, double* x, acc_t* u) {
    for (int64_t j = 0; j < A->n; ++j) u[j] = 0;
    for (int64_t i = r0; i < r1; ++i) {
        const double r = row_dot(A->rowptr, A->col, A->val, i, x); /* <a^i, x>, L41 */
        double c = violation(r, lb[i], ub[i]);
        if (c != 0.0) {
            double y = (d[i] * dscale) * c;
            for (int64_t k = A->rowptr[i]; k < A->rowptr[i + 1]; ++k) u[A->col[k]] += (acc_t)A->val[k] * y;
        }
    }
    for (int64_t j = 0; j < A->n; ++j) {
        double t = x[j] - lambda * (double)u[j]; /* Eq. 3 (L46) */
        if (t < lo[j]) t = lo[j];        /* BoxProjection, L427 */
        if (t > hi[j]) t = hi[j];
        x[j] = t;
    }
}

void orc_sweep(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* lb,
               const double* ub, const double* d, const double* lo, const double* hi, double lambda, double* x) {
    csr_t A = {m, n, rowptr, col, val};
    acc_t* u = (acc_t*)malloc(sizeof(acc_t) * (size_t)n);
    sweep_rows(&A, 0, m, lb, ub, d, 1.0, lo, hi, lambda, x, u);
    free(u);
}

/* ---- O-BLOCK-SWEEP (block-iterative family; A-14): blocks of contiguous rows visited in
 * index order; within block t a simultaneous step with weights w_i / W_t, W_t = sum_{i in B_t} w_i;
 * box after every block. */
void orc_block_sweep(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val,
                     const double* lb, const double* ub, const double* w, const double* d, const double* lo,
                     const double* hi, double lambda, int n_blocks, const int64_t* block_rowptr, double* x) {
    csr_t A = {m, n, rowptr, col, val};
    acc_t* u = (acc_t*)malloc(sizeof(acc_t) * (size_t)n);
    for (int t = 0; t < n_blocks; ++t) {
        acc_t W_acc = 0;
        for (int64_t i = block_rowptr[t]; i < block_rowptr[t + 1]; ++i) W_acc += w[i];
        const double W = (double)W_acc;
        if (!(W > 0.0)) continue;
        sweep_rows(&A, block_rowptr[t], block_rowptr[t + 1], lb, ub, d, 1.0 / W, lo, hi, lambda, x, u);
    }
    free(u);
}

/* ---- O-DROP: Table A.5 row 1, x^{k+1} = x^k - Z A^T M (A x^k - b) with M = diag(w_i), sum w_i = 1, and
 * Z = diag(1 / nnz(A_{:,j})) (caption, L608; A-19: M is per row, Z per column; a column without stored entries gets
 * z_j = 0).  Reading A-26: the residual (A x - b)_i is the hyperslab violation c_i(x) -- for an equality row
 * lb_i = ub_i = b_i that IS <a^i,x> - b_i, which is the case the table prints -- the relaxation lambda multiplies the
 * step (lambda = 1 is the table's formula) and the box follows the step as in every other sweep (L427, A-2). */
void orc_drop_sweep(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* lb,
                    const double* ub, const double* w, const double* lo, const double* hi, double lambda, double* x) {
    acc_t* u = (acc_t*)malloc(sizeof(acc_t) * (size_t)n);
    int64_t* cnt = (int64_t*)calloc((size_t)n, sizeof(int64_t));
    for (int64_t k = 0; k < rowptr[m]; ++k) cnt[col[k]]++; /* nnz(A_{:,j}): stored entries of column j */
    for (int64_t j = 0; j < n; ++j) u[j] = 0;
    for (int64_t i = 0; i < m; ++i) {
        const double r = row_dot(rowptr, col, val, i, x);
        const double c = violation(r, lb[i], ub[i]);
        if (c != 0.0) {
            const double y = w[i] * c; /* M (A x - b) */
            for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) u[col[k]] += (acc_t)val[k] * y;
        }
    }
    for (int64_t j = 0; j < n; ++j) {
        const double z = cnt[j] > 0 ? 1.0 / (double)cnt[j] : 0.0;
        double t = x[j] - lambda * (z * (double)u[j]);
        if (t < lo[j]) t = lo[j];
        if (t > hi[j]) t = hi[j];
        x[j] = t;
    }
    free(u);
    free(cnt);
}

/* ---- O-EMR: Table A.5 row 4, Landweber with error-minimising relaxation:
 *   p = A^T M (A x - b),   x^{k+1} = x^k - ( ||p||^2 / ||M^{1/2} A p||^2 ) p,   M = diag(w_i) (L608).
 * For equality rows the factor is the exact minimiser of ||M^{1/2}(A(x - t p) - b)||^2 over t (pinned by that).  A-26 as
 * for DROP: residual = hyperslab violation, box after the step.  A zero denominator (p = 0 or A p = 0) leaves x as it is.
 * step_out (optional) receives the factor. */
void orc_emr_sweep(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, const double* lb,
                   const double* ub, const double* w, const double* lo, const double* hi, double* x, double* step_out) {
    acc_t* u = (acc_t*)malloc(sizeof(acc_t) * (size_t)n);
    double* p = (double*)malloc(sizeof(double) * (size_t)n);
    for (int64_t j = 0; j < n; ++j) u[j] = 0;
    for (int64_t i = 0; i < m; ++i) {
        const double r = row_dot(rowptr, col, val, i, x);
        const double c = violation(r, lb[i], ub[i]);
        if (c != 0.0) {
            const double y = w[i] * c;
            for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) u[col[k]] += (acc_t)val[k] * y;
        }
    }
    acc_t pp = 0, qq = 0;
    for (int64_t j = 0; j < n; ++j) {
        p[j] = (double)u[j];
        pp += (acc_t)p[j] * p[j];
    }
    for (int64_t i = 0; i < m; ++i) {
        const double q = row_dot(rowptr, col, val, i, p); /* (A p)_i */
        qq += (acc_t)(w[i] * q) * q;
    }
    const double num = (double)pp, den = (double)qq;
    const double t = den > 0.0 ? num / den : 0.0;
    if (step_out) *step_out = t;
    for (int64_t j = 0; j < n; ++j) {
        double v = x[j] - t * p[j];
        if (v < lo[j]) v = lo[j];
        if (v > hi[j]) v = hi[j];
        x[j] = v;
    }
    free(u);
    free(p);
}

/* ---- O-PROX.  delta_i = |c_i| / ||a^i|| = Euclidean distance to C_i (0 for empty rows, A-4/A-5).
 * mode 0: 1/2 sum w_i delta_i^2 (Eq. 5); mode 1: sum w_i delta_i^p (Eq. 12);
 * mode 2: max_i delta_i (Eq. 13). */
double orc_proximity(int64_t m, const int64_t* rowptr, const int32_t* col, const double* val, const double* lb,
                     const double* ub, const double* w, const double* rho, const double* x, int mode, double p) {
    acc_t acc = 0;
    double mx = 0.0;
    for (int64_t i = 0; i < m; ++i) {
        const double r = row_dot(rowptr, col, val, i, x);
        double c = violation(r, lb[i], ub[i]);
        double delta = rho[i] > 0.0 ? fabs(c) / sqrt(rho[i]) : 0.0;
        if (mode == 0) acc += (w[i] * delta) * delta;
        else if (mode == 1) acc += w[i] * pow(delta, p);
        else if (delta > mx) mx = delta;
    }
    if (mode == 2) return mx;
    return mode == 0 ? 0.5 * (double)acc : (double)acc;
}

/* ---- objectives ---------------------------------------------------------------------------------- */
/* TV2D, Eq. 15 on an ny x nx row-major image X[i*nx+j]: terms only for i < ny-1, j < nx-1. */
double orc_tv2d(const double* X, int64_t ny, int64_t nx) {
    acc_t s = 0;
    for (int64_t i = 0; i + 1 < ny; ++i)
        for (int64_t j = 0; j + 1 < nx; ++j) {
            double dx = X[(i + 1) * nx + j] - X[i * nx + j];
            double dy = X[i * nx + j + 1] - X[i * nx + j];
            s += sqrt(dx * dx + dy * dy);
        }
    return (double)s;
}

/* Gradient of Eq. 15 as printed, term by term (A-8); a term with t = 0 contributes 0 (A-9).  A pixel receives at most
 * three contributions, in the order of this loop: +dx/t of term (i-1,j), +dy/t of term (i,j-1), -(dx+dy)/t of its own
 * term (i,j): g_ij = ((0 + a) + b) - c in fp64. */
void orc_tv2d_grad(const double* X, int64_t ny, int64_t nx, double* g) {
    for (int64_t q = 0; q < ny * nx; ++q) g[q] = 0.0;
    for (int64_t i = 0; i + 1 < ny; ++i)
        for (int64_t j = 0; j + 1 < nx; ++j) {
            double dx = X[(i + 1) * nx + j] - X[i * nx + j];
            double dy = X[i * nx + j + 1] - X[i * nx + j];
            double t = sqrt(dx * dx + dy * dy);
            if (t > 0.0) {
                g[i * nx + j] -= (dx + dy) / t;
                g[(i + 1) * nx + j] += dx / t;
                g[i * nx + j + 1] += dy / t;
            }
        }
}

/* TV1D (A-16): f = sum_{i<n-1} |x_{i+1} - x_i|, subgradient with sgn(0) = 0. */
double orc_tv1d(const double* x, int64_t n) {
    acc_t s = 0;
    for (int64_t i = 0; i + 1 < n; ++i) s += fabs(x[i + 1] - x[i]);
    return (double)s;
}
void orc_tv1d_grad(const double* x, int64_t n, double* g) {
    for (int64_t i = 0; i < n; ++i) g[i] = 0.0;
    for (int64_t i = 0; i + 1 < n; ++i) {
        double dlt = x[i + 1] - x[i];
        double s = (dlt > 0.0) - (dlt < 0.0);
        g[i] -= s;
        g[i + 1] += s;
    }
}

/* TV3D: Eq. 15 with a third difference (north_star: "2D/3D TV-gradient stencil"; reading A-27): on an
 * nz x ny x nx volume X[(i*ny+j)*nx+k], terms for i < nz-1, j < ny-1, k < nx-1 only,
 *   t_ijk = sqrt( (X_{i+1,j,k}-X_ijk)^2 + (X_{i,j+1,k}-X_ijk)^2 + (X_{i,j,k+1}-X_ijk)^2 ). */
double orc_tv3d(const double* X, int64_t nz, int64_t ny, int64_t nx) {
    acc_t s = 0;
    for (int64_t i = 0; i + 1 < nz; ++i)
        for (int64_t j = 0; j + 1 < ny; ++j)
            for (int64_t k = 0; k + 1 < nx; ++k) {
                const int64_t p = (i * ny + j) * nx + k;
                double dz = X[p + ny * nx] - X[p], dy = X[p + nx] - X[p], dx = X[p + 1] - X[p];
                s += sqrt((dz * dz + dy * dy) + dx * dx);
            }
    return (double)s;
}
/* gradient term by term as in orc_tv2d_grad (A-8, A-9): a voxel receives +dz/t of term (i-1,j,k), +dy/t of (i,j-1,k),
 * +dx/t of (i,j,k-1) and -(dz+dy+dx)/t of its own term, in the order the loop meets them. */
void orc_tv3d_grad(const double* X, int64_t nz, int64_t ny, int64_t nx, double* g) {
    for (int64_t q = 0; q < nz * ny * nx; ++q) g[q] = 0.0;
    for (int64_t i = 0; i + 1 < nz; ++i)
        for (int64_t j = 0; j + 1 < ny; ++j)
            for (int64_t k = 0; k + 1 < nx; ++k) {
                const int64_t p = (i * ny + j) * nx + k;
                double dz = X[p + ny * nx] - X[p], dy = X[p + nx] - X[p], dx = X[p + 1] - X[p];
                double t = sqrt((dz * dz + dy * dy) + dx * dx);
                if (t > 0.0) {
                    g[p] -= ((dz + dy) + dx) / t;
                    g[p + ny * nx] += dz / t;
                    g[p + nx] += dy / t;
                    g[p + 1] += dx / t;
                }
            }
}

/* MEAN: f_Mean(d) = (1/N_S) sum_{i in S} d_i with d = D_S x (Eq. 21); D_S is the md x n CSR of the
 * structure's voxels (md = N_S).  Gradient (1/N_S) D_S^T 1, constant in x. */
double orc_mean(int64_t md, const int64_t* rowptr, const int32_t* col, const double* val, const double* x) {
    acc_t s = 0;
    for (int64_t i = 0; i < md; ++i) s += row_dot(rowptr, col, val, i, x);
    return (double)s / (double)md;
}
void orc_mean_grad(int64_t md, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val, double* g) {
    acc_t* u = (acc_t*)malloc(sizeof(acc_t) * (size_t)n);
    for (int64_t j = 0; j < n; ++j) u[j] = 0;
    for (int64_t i = 0; i < md; ++i)
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) u[col[k]] += val[k];
    for (int64_t j = 0; j < n; ++j) g[j] = (double)u[j] / (double)md;
    free(u);
}

/* DOSE (A-15): f = ||D x||^2, g = 2 D^T (D x); D is md x n CSR. */
double orc_dose(int64_t md, const int64_t* rowptr, const int32_t* col, const double* val, const double* x) {
    acc_t s = 0;
    for (int64_t i = 0; i < md; ++i) {
        const double r = row_dot(rowptr, col, val, i, x);
        s += (acc_t)r * r;
    }
    return (double)s;
}
void orc_dose_grad(int64_t md, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val,
                   const double* x, double* g) {
    acc_t* u = (acc_t*)malloc(sizeof(acc_t) * (size_t)n); /* u = D^T (D x) */
    for (int64_t j = 0; j < n; ++j) u[j] = 0;
    for (int64_t i = 0; i < md; ++i) {
        const double r = row_dot(rowptr, col, val, i, x);
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k) u[col[k]] += (acc_t)val[k] * r;
    }
    for (int64_t j = 0; j < n; ++j) g[j] = 2.0 * (double)u[j];
    free(u);
}

/* objective descriptor: kind 0 = none (f = 0, g = 0), 1 = TV2D (ny, nx), 2 = TV1D, 3 = DOSE, 4 = MEAN (Eq. 21),
 * 5 = TV3D (nz, ny, nx) */
typedef struct {
    int kind;
    int64_t ny, nx;
    int64_t md;
    const int64_t* d_rowptr;
    const int32_t* d_col;
    const double* d_val;
    int64_t nz; /* TV3D only */
} obj_t;

static double obj_value(const obj_t* O, int64_t n, const double* x) {
    switch (O->kind) {
        case 1: return orc_tv2d(x, O->ny, O->nx);
        case 2: return orc_tv1d(x, n);
        case 3: return orc_dose(O->md, O->d_rowptr, O->d_col, O->d_val, x);
        case 4: return orc_mean(O->md, O->d_rowptr, O->d_col, O->d_val, x);
        case 5: return orc_tv3d(x, O->nz, O->ny, O->nx);
        default: return 0.0;
    }
}
static void obj_grad(const obj_t* O, int64_t n, const double* x, double* g) {
    switch (O->kind) {
        case 1: orc_tv2d_grad(x, O->ny, O->nx, g); break;
        case 2: orc_tv1d_grad(x, n, g); break;
        case 3: orc_dose_grad(O->md, n, O->d_rowptr, O->d_col, O->d_val, x, g); break;
        case 4: orc_mean_grad(O->md, n, O->d_rowptr, O->d_col, O->d_val, g); break;
        case 5: orc_tv3d_grad(x, O->nz, O->ny, O->nx, g); break;
        default: for (int64_t j = 0; j < n; ++j) g[j] = 0.0;
    }
}

/* ---- O-PERTURB: the perturbation phase, Algorithm 1 lines 4-17.
 *  fx <- f(x); for n = 0..N-1: g <- grad f(x^{k,n}) (A-7: recomputed at every reduction step);
 *  v <- -g/||g|| (A-6: minus sign per L84/L93; v = 0 if ||g|| = 0);
 *  trial loop: beta <- beta0 * a^l (A-10; A-20: a^l is the running fp64 product a_pow(l), not libm pow),
 *  z <- x + beta v, l <- l+1,
 *  accept iff f(z) <= f(x^{k,n}) (L149, A-11).  J_max trials per step (A-12).
 *  policy 0 = PER_TRIAL: one persistent counter *ell, incremented on every trial, never reset.
 *  policy 1 = PER_SWEEP: beta_{k,j} = beta0 * a^{k+j}, j reset to 0 at every reduction step (literal Alg. 1).
 *  decisions/n_dec: optional log of every trial (1 accept / 0 reject), capacity cap_dec.
 *  forced: optional replay of a decision sequence (A-13 trace-replay); NULL = decide by the test.
 *  margins: optional per-trial |fz-fx|/max(1,|fx|).  Returns number of trials; *warn |= 1 if J_max hit. */
#define J_MAX 10000
/* a^e by e successive fp64 multiplications starting from 1 (A-20): every implementation of IEEE-754 gets the same
 * bits, which libm pow() does not promise. */
static double a_pow(double a, int64_t e) {
    double p = 1.0;
    for (int64_t q = 0; q < e; ++q) p *= a;
    return p;
}
int64_t orc_perturb(int64_t n, const obj_t* O, double* x, int64_t* ell, int64_t k, int N, double beta0, double a,
                    int policy, double* g, double* z, int8_t* decisions, double* margins, int64_t cap_dec,
                    int64_t* n_dec, const int8_t* forced, int* warn, double* fx_out) {
    double fx = obj_value(O, n, x);
    int64_t trials = 0;
    for (int nred = 0; nred < N; ++nred) {
        obj_grad(O, n, x, g);
        acc_t s_acc = 0;
        for (int64_t j = 0; j < n; ++j) s_acc += (acc_t)g[j] * g[j];
        const double s = sqrt((double)s_acc);
        int64_t jloc = 0;
        int accepted = 0;
        double apow = a_pow(a, policy == 0 ? *ell : k); /* a^l resp. a^(k+0) */
        for (int trial = 0; trial < J_MAX && !accepted; ++trial) {
            double beta = beta0 * apow;
            apow *= a;
            for (int64_t j = 0; j < n; ++j) z[j] = s > 0.0 ? x[j] + beta * (-g[j] / s) : x[j];
            (*ell)++;
            jloc++;
            trials++;
            double fz = obj_value(O, n, z);
            int acc = forced ? (int)forced[*n_dec] : (fz <= fx);
            if (decisions && *n_dec < cap_dec) {
                decisions[*n_dec] = (int8_t)acc;
                if (margins) margins[*n_dec] = fabs(fz - fx) / fmax(1.0, fabs(fx));
            }
            (*n_dec)++;
            if (acc) {
                memcpy(x, z, sizeof(double) * (size_t)n);
                fx = fz;
                accepted = 1;
            }
        }
        if (!accepted && warn) *warn |= 1; /* A-12: step skipped */
    }
    if (fx_out) *fx_out = fx;
    return trials;
}

/* ---- O-PERTURB-ADAPTIVE: the perturbation phase with the subgradient-projection step size of Eq. 11
 * ("Nikazad et al. [7]"):
 *      beta = 0                          if f(x) <= f_ref,
 *      beta = (f(x) - f_ref) / ||g_f(x)||  if f(x) >  f_ref,
 * used in Eq. 10 with v = -g/||g|| (A-6), i.e. x <- x - ((f(x) - f_ref)/||g||^2) g: the projection of x onto the half-space
 * {y : f(x) + <g, y - x> <= f_ref}.  Eq. 11 DEFINES beta, so there is no trial loop, no accept test and no exponent l
 * (reading A-30); N such steps per phase (N = 1 is the literal Eq. 10), each with f and g re-evaluated (A-7); a step with
 * ||g|| = 0 is beta = 0.
 * f_ref "is automatically updated throughout the iterations" (L108) by a rule the paper only cites.  Reading A-30 -- the
 * part of this function that is PARITY UNPINNED against the paper (the rule is ours; the step itself is pinned):
 *      if the phase started at a point with f(x^k) <= f_ref, then after the phase f_ref <- shrink * f(x^k), shrink in (0, 1]
 *      (the iterate has reached the reference, so the reference is moved below it); otherwise f_ref is kept.
 * decisions/n_dec: optional log, 1 = a step with beta > 0 was taken, 0 = beta = 0.  Returns the number of steps with beta > 0. */
int64_t orc_perturb_adaptive(int64_t n, const obj_t* O, double* x, int N, double* f_ref, double shrink, double* g,
                             int8_t* decisions, int64_t cap_dec, int64_t* n_dec, double* fx_out) {
    const double f_start = obj_value(O, n, x);
    double fx = f_start;
    int64_t steps = 0;
    for (int nred = 0; nred < N; ++nred) {
        if (nred > 0) fx = obj_value(O, n, x);
        obj_grad(O, n, x, g);
        acc_t s_acc = 0;
        for (int64_t j = 0; j < n; ++j) s_acc += (acc_t)g[j] * g[j];
        const double s = sqrt((double)s_acc);
        const int take = fx > *f_ref && s > 0.0;
        if (take) {
            const double beta = (fx - *f_ref) / s; /* Eq. 11 */
            for (int64_t j = 0; j < n; ++j) x[j] = x[j] + beta * (-g[j] / s); /* Eq. 10's perturbation, v = -g/||g|| */
            steps++;
        }
        if (decisions && *n_dec < cap_dec) decisions[*n_dec] = (int8_t)take;
        (*n_dec)++;
    }
    if (f_start <= *f_ref) *f_ref = shrink * f_start;
    if (fx_out) *fx_out = fx; /* f at the point the last step started from */
    return steps;
}

/* ---- O-SUPERIORIZE: Algorithm 1, Eq. 10 (L91): for each sweep k the perturbation
 * phase comes first, then the feasibility-seeking operator T.  Runs sweeps k0 .. k0+n_iter-1 so that a caller can
 * take snapshots between calls (state = x, ell, k).
 * trace[k-k0][0..3] = {proximity mode 0 after the sweep, f(x) after the sweep, #trials, ell}.
 *
 * run_opt_t selects T and the stopping rule:
 *   algorithm 0: simultaneous sweep (A-1), 1: block-iterative (A-14; needs n_blocks), 2: DROP, 3: EMR (Table A.5).
 *   stop_enabled: the paper's default termination (section 2.2.1, L239-243 section 2.2.3), reading A-25:
 *     P^k = Eq. 12 with the default p = 2 at the iterate x^k (the point after sweep k-1; P^0 at the starting point),
 *     f^k = f(x^k);
 *     (1) P^k <= prox_tol;
 *     (2) dP = |P^k - P^{k-1}| / max(1, P^{k-1}) < dprox_tol for n_consec consecutive iterations;
 *     (f) df = |f^k - f^{k-1}| / max(1, f^{k-1}) < dobj_tol                       (superiorized runs only);
 *     stop iff ((1) or (2)) [and (f) when an objective is perturbed]; criterion (3), N_max, is n_iter.
 *     The test is made after every sweep except the last of the call (which returns anyway), so *n_done < n_iter
 *     exactly when a criterion fired; *stop_reason = 1*(1) + 2*(2) + 4*(f) at that point, else 0. */
typedef struct {
    int algorithm;
    int stop_enabled;
    double prox_tol, dprox_tol;
    int n_consec;
    double dobj_tol;
    int64_t n_restart;
    int64_t nz; /* TV3D: shape = (nz, ny, nx) */
    int step_rule;       /* 0: power law beta0 * a^l with the accept test (Alg. 1); 1: Eq. 11 (O-PERTURB-ADAPTIVE, A-30) */
    double f_ref;        /* Eq. 11's reference value; UPDATED IN PLACE by the run (A-30) */
    double f_ref_shrink; /* A-30's update factor */
} run_opt_t;

int orc_superiorize_ex(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val,
                       const double* lb, const double* ub, const double* w, const double* rho, const double* d,
                       const double* lo, const double* hi, double lambda, int n_blocks, const int64_t* block_rowptr,
                       int obj_kind, int64_t ny, int64_t nx, int64_t md, const int64_t* d_rowptr, const int32_t* d_col,
                       const double* d_val, double* x, int64_t* ell, int64_t k0, int n_iter, int N, double beta0,
                       double a, int policy, double* trace, int8_t* decisions, double* margins, int64_t cap_dec,
                       int64_t* n_dec, const int8_t* forced, run_opt_t* opt, int* n_done, int* stop_reason) {
    obj_t O = {obj_kind, ny, nx, md, d_rowptr, d_col, d_val, opt->nz};
    double* g = (double*)malloc(sizeof(double) * (size_t)n);
    double* z = (double*)malloc(sizeof(double) * (size_t)n);
    int warn = 0;
    const int perturbed = N > 0 && obj_kind != 0;
    double P_prev = 0.0, f_prev = 0.0;
    int consec = 0;
    if (opt->stop_enabled) {
        P_prev = orc_proximity(m, rowptr, col, val, lb, ub, w, rho, x, 1, 2.0); /* P^0, Eq. 12 with p = 2 */
        f_prev = obj_value(&O, n, x);
    }
    if (n_done) *n_done = 0;
    if (stop_reason) *stop_reason = 0;
    for (int it = 0; it < n_iter; ++it) {
        int64_t k = k0 + it;
        int64_t trials = 0;
        /* restarted perturbations ("l was restarted after every 50 iterations"; A-24): at the start of
         * sweep k = r * n_restart, r = 1, 2, ..., the exponent is reset to r ("l = 1 after the first restart, l = 2 after
         * the second"), which keeps sum beta finite: cycle r contributes at most beta0 a^r / (1 - a). */
        if (opt->n_restart > 0 && k > 0 && k % opt->n_restart == 0) *ell = k / opt->n_restart;
        if (perturbed && opt->step_rule == 1)
            trials = orc_perturb_adaptive(n, &O, x, N, &opt->f_ref, opt->f_ref_shrink, g, decisions, cap_dec, n_dec, NULL);
        else if (perturbed)
            trials = orc_perturb(n, &O, x, ell, k, N, beta0, a, policy, g, z, decisions, margins, cap_dec, n_dec,
                                 forced, &warn, NULL);
        switch (opt->algorithm) {
            case 1: orc_block_sweep(m, n, rowptr, col, val, lb, ub, w, d, lo, hi, lambda, n_blocks, block_rowptr, x); break;
            case 2: orc_drop_sweep(m, n, rowptr, col, val, lb, ub, w, lo, hi, lambda, x); break;
            case 3: orc_emr_sweep(m, n, rowptr, col, val, lb, ub, w, lo, hi, x, NULL); break;
            default: orc_sweep(m, n, rowptr, col, val, lb, ub, d, lo, hi, lambda, x);
        }
        if (trace) {
            trace[4 * it + 0] = orc_proximity(m, rowptr, col, val, lb, ub, w, rho, x, 0, 2.0);
            trace[4 * it + 1] = obj_value(&O, n, x);
            trace[4 * it + 2] = (double)trials;
            trace[4 * it + 3] = (double)(*ell);
        }
        if (n_done) *n_done = it + 1;
        if (opt->stop_enabled && it + 1 < n_iter) {
            const double P = orc_proximity(m, rowptr, col, val, lb, ub, w, rho, x, 1, 2.0);
            const double f = obj_value(&O, n, x);
            const int c1 = P <= opt->prox_tol;
            const double dP = fabs(P - P_prev) / fmax(1.0, P_prev);
            consec = dP < opt->dprox_tol ? consec + 1 : 0;
            const int c2 = consec >= opt->n_consec;
            const double df = fabs(f - f_prev) / fmax(1.0, f_prev);
            const int cf = df < opt->dobj_tol;
            P_prev = P;
            f_prev = f;
            if ((c1 || c2) && (!perturbed || cf)) {
                if (stop_reason) *stop_reason = c1 + 2 * c2 + 4 * (perturbed && cf);
                break;
            }
        }
    }
    free(g);
    free(z);
    return warn;
}

int orc_superiorize(int64_t m, int64_t n, const int64_t* rowptr, const int32_t* col, const double* val,
                    const double* lb, const double* ub, const double* w, const double* rho, const double* d,
                    const double* lo, const double* hi, double lambda, int n_blocks, const int64_t* block_rowptr,
                    int obj_kind, int64_t ny, int64_t nx, int64_t md, const int64_t* d_rowptr, const int32_t* d_col,
                    const double* d_val, double* x, int64_t* ell, int64_t k0, int n_iter, int N, double beta0,
                    double a, int policy, double* trace, int8_t* decisions, double* margins, int64_t cap_dec,
                    int64_t* n_dec, const int8_t* forced, int64_t n_restart) {
    run_opt_t opt = {n_blocks > 0 ? 1 : 0, 0, 0.0, 0.0, 0, 0.0, n_restart, 0, 0, 0.0, 0.0};
    return orc_superiorize_ex(m, n, rowptr, col, val, lb, ub, w, rho, d, lo, hi, lambda, n_blocks, block_rowptr, obj_kind,
                              ny, nx, md, d_rowptr, d_col, d_val, x, ell, k0, n_iter, N, beta0, a, policy, trace,
                              decisions, margins, cap_dec, n_dec, forced, &opt, NULL, NULL);
}

/* stand-alone perturbation phase (what sup_perturb_tv / sup_perturb_dose are checked against) */
int64_t orc_perturb_phase(int64_t n, int obj_kind, int64_t ny, int64_t nx, int64_t md, const int64_t* d_rowptr,
                          const int32_t* d_col, const double* d_val, double* x, int64_t* ell, int64_t k, int N,
                          double beta0, double a, int policy, int8_t* decisions, double* margins, int64_t cap_dec,
                          int64_t* n_dec, const int8_t* forced, int* warn, double* fx_out) {
    obj_t O = {obj_kind, ny, nx, md, d_rowptr, d_col, d_val, 0};
    double* g = (double*)malloc(sizeof(double) * (size_t)n);
    double* z = (double*)malloc(sizeof(double) * (size_t)n);
    int64_t t = orc_perturb(n, &O, x, ell, k, N, beta0, a, policy, g, z, decisions, margins, cap_dec, n_dec, forced,
                            warn, fx_out);
    free(g);
    free(z);
    return t;
}

/* the same for objectives that need the third shape entry (TV3D: nz, ny, nx) */
int64_t orc_perturb_phase3(int64_t n, int obj_kind, int64_t nz, int64_t ny, int64_t nx, double* x, int64_t* ell, int64_t k,
                           int N, double beta0, double a, int policy, int8_t* decisions, double* margins, int64_t cap_dec,
                           int64_t* n_dec, const int8_t* forced, int* warn, double* fx_out) {
    obj_t O = {obj_kind, ny, nx, 0, NULL, NULL, NULL, nz};
    double* g = (double*)malloc(sizeof(double) * (size_t)n);
    double* z = (double*)malloc(sizeof(double) * (size_t)n);
    int64_t t = orc_perturb(n, &O, x, ell, k, N, beta0, a, policy, g, z, decisions, margins, cap_dec, n_dec, forced,
                            warn, fx_out);
    free(g);
    free(z);
    return t;
}

/* stand-alone adaptive phase (what sup_perturb_adaptive is checked against); nz = 0 unless TV3D */
int64_t orc_perturb_adaptive_phase(int64_t n, int obj_kind, int64_t nz, int64_t ny, int64_t nx, int64_t md,
                                   const int64_t* d_rowptr, const int32_t* d_col, const double* d_val, double* x, int N,
                                   double* f_ref, double shrink, int8_t* decisions, int64_t cap_dec, int64_t* n_dec,
                                   double* fx_out) {
    obj_t O = {obj_kind, ny, nx, md, d_rowptr, d_col, d_val, nz};
    double* g = (double*)malloc(sizeof(double) * (size_t)n);
    int64_t t = orc_perturb_adaptive(n, &O, x, N, f_ref, shrink, g, decisions, cap_dec, n_dec, fx_out);
    free(g);
    return t;
}
