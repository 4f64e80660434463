// sup_perturb.cu -- S5-S7 of the hot path: the perturbation phase of Algorithm 1
// as ONE persistent cooperative kernel per phase.
//
//   fx <- f(x)
//   for n = 0..N-1:  g <- grad f(x^{k,n}) (A-7), s <- ||g||_2, v = -g/s (A-6)
//        trial loop:  beta <- beta0 * a^l (A-10; a^l is the running fp64 product, A-20), z <- x + beta v, l <- l+1,
//                     accept iff f(z) <= f(x^{k,n}) (L149, A-11); at most J_max trials (A-12)
//
// The number of trials is data dependent, so the loop lives on the device: all CTAs of the grid are co-resident
// (cooperative launch) and meet after every pass at a grid barrier that is fused with the second stage of the
// reduction -- the last CTA to arrive sums the per-CTA partials in a fixed order and publishes the totals with the
// barrier's generation flip, so every CTA takes the accept decision from the same numbers: no host round trip, and
// the launch is capturable in a CUDA graph.  z is never stored on its own: z_p = round_T(x_p - (beta/s) g_p) is
// recomputed wherever it is needed.
//
// TV objectives (TV2D: Eq. 15, gradient A-8; TV3D: the same with a third difference, A-27; TV1D: A-16): the
// gradient pass of a tile computes every term t_p of the tile anyway, so f comes for free with it.  One pass therefore
// evaluates the FIRST candidate step of a reduction step completely -- z, f(z), grad f(z), ||grad f(z)||^2 -- and when
// that candidate is accepted (the common case once beta is small) the next reduction step can start at once:
// 1 + N grid-wide passes per phase instead of 1 + 2N.  A rejected first candidate falls back to evaluating the next
// SUP_TRIAL_BATCH candidates per pass, decided strictly in order: the trial / decision / l sequence is exactly
// Algorithm 1's.  The dose objective ||D x||^2 (A-15) and f_Mean run as launch sequences on the product kernels (sup_algos.cu).
// Objective terms, norms and beta are fp64 in both modes.
#include <math.h>
#include <stdlib.h>

#include "sup_internal.cuh"
#include "sup_perturb_args.cuh"

#define TILE_H 16
#define TILE_W 64
#define BARRIER_SPIN_LIMIT (1u << 24)
#define SUP_TRIAL_BATCH 8  // candidate steps evaluated per pass after a rejected first candidate (TV objectives)


// ---- grid barrier (all CTAs co-resident by cooperative launch) ----------------------------------------------
// Grid barrier fused with the second stage of a reduction.  On entry v[0..NV) are this THREAD's shares; every CTA sums its threads'
// shares, stores the NV sums to its slots of the partials buffer and adds 1 to a MONOTONE arrival counter (a release: the partials
// are visible before the count).  Then EVERY CTA waits until the counter has reached this barrier's target (an acquire) and adds the
// partials of all CTAs itself, in the same fixed order -- the same numbers in the same order give the same bits in every CTA, which
// is what keeps the kernel's control flow uniform.  Three L2 round trips per barrier (arrive, see the target, read the partials)
// against four when the last CTA to arrive added the partials and published totals (arrive with the old value returned, read
// partials, release a flag, read totals): 4.4 -> ~3.3 us at 256 CTAs (profiles/r02c).  The counter is never reset inside a launch;
// a launch starts from st->bar_base, which CTA 0 of the launch before left there (a CTA reads it before its first arrival, and CTA 0
// can only reach the end of a kernel after every CTA has arrived at its barriers).  The partials are double-buffered by barrier
// parity: a CTA writes the buffer of barrier i + 2 only after barrier i + 1, which every CTA reaches after reading barrier i's.
// On return v[] holds the totals in every thread.  Returns false after a time-out (fault bit 0 is set): the caller leaves the
// kernel instead of computing on inconsistent partials.
template <int NV>
__device__ __forceinline__ void cta_sum_batch(double* v);
__device__ __forceinline__ void red_release_add(unsigned long long* p, unsigned long long v) {
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

struct GridBar {
    unsigned long long target;  // value of the arrival counter when the barrier last passed is complete
    unsigned n;                 // barriers passed in this launch (parity selects the partials buffer)
};

template <int NV>
__device__ __forceinline__ bool grid_reduce(DevState* st, double* partials, int stride, double* v, GridBar& gb) {
    __shared__ int s_ok;
    cta_sum_batch<NV>(v);
    gb.target += gridDim.x;
    double* buf = partials + (gb.n & 1u) * SUP_MAX_PARTIALS;
    gb.n += 1u;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < NV; ++b) buf[b * stride + blockIdx.x] = v[b];
        red_release_add(&st->bar_count, 1ull);
        int ok = 1;
        unsigned spins = 0;
        while (ld_acquire(&st->bar_count) < gb.target) {
            __nanosleep(20);
            if (++spins > BARRIER_SPIN_LIMIT) {
                atomicOr(&st->fault, 1);
                ok = 0;
                break;
            }
        }
        s_ok = ok;
    }
    __syncthreads();
    if (!s_ok) return false;
    double w[NV];
#pragma unroll
    for (int b = 0; b < NV; ++b) {
        w[b] = 0.0;
        for (int q = threadIdx.x; q < int(gridDim.x); q += SUP_THREADS) w[b] += __ldcg(buf + b * stride + q);
    }
    cta_sum_batch<NV>(w);
#pragma unroll
    for (int b = 0; b < NV; ++b) v[b] = w[b];
    return true;
}

// sum over the CTA, result valid in every thread; fixed order
__device__ __forceinline__ double cta_sum(double v) {
    __shared__ double ws[SUP_THREADS / 32];
    __shared__ double tot;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) ws[wid] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int q = 0; q < SUP_THREADS / 32; ++q) t += ws[q];
        tot = t;
    }
    __syncthreads();
    return tot;
}

// B sums at once (same order per value as cta_sum)
template <int B>
__device__ __forceinline__ void cta_sum_batch(double* v) {
    __shared__ double wsb[B][SUP_THREADS / 32];
    __shared__ double totb[B];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int b = 0; b < B; ++b)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[b] += __shfl_xor_sync(0xffffffffu, v[b], o);
    __syncthreads();
    if (lane == 0)
#pragma unroll
        for (int b = 0; b < B; ++b) wsb[b][wid] = v[b];
    __syncthreads();
    if (threadIdx.x < B) {
        double t = 0.0;
        for (int q = 0; q < SUP_THREADS / 32; ++q) t += wsb[threadIdx.x][q];
        totb[threadIdx.x] = t;
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < B; ++b) v[b] = totb[b];
}

template <typename T>
__device__ __forceinline__ double zval(const T* __restrict__ x, const T* __restrict__ g, double coef, int64_t p) {
    const double xv = double(__ldcg(x + p));
    if (coef == 0.0) return xv;
    return double(T(fma(-coef, double(__ldcg(g + p)), xv)));  // z rounded to the storage type, as it would be stored
}

// sqrt(d) and 1/sqrt(d) for the TV terms via rsqrt (1 ulp, a short MUFU + Newton chain) instead of IEEE sqrt and
// divide, whose dependent fp64 sequences were the latency of every phase of this kernel: t = d * rsqrt(d) is within
// 2 ulp of sqrt(d), far inside the fp64 parity bar (1e-10) and the knife-edge threshold of the accept test (1e-12).
__device__ __forceinline__ double tv_norm(double d) { return d > 0.0 ? d * rsqrt(d) : 0.0; }

// ---- objective value of z = x - coef g : this thread's share (not yet reduced) ------------------------------
template <typename T>
__device__ double tv2d_share(const PArgs<T>& A, double coef) {
    // Eq. 15: terms for i < ny-1, j < nx-1 only
    const int64_t h = A.ny - 1, w = A.nx - 1;
    const int64_t total = h > 0 && w > 0 ? h * w : 0;
    double acc = 0.0;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < total; q += int64_t(gridDim.x) * blockDim.x) {
        const int64_t i = q / w, j = q - i * w;
        const int64_t p = i * A.nx + j;
        const double z00 = zval(A.x, A.g, coef, p), z10 = zval(A.x, A.g, coef, p + A.nx), z01 = zval(A.x, A.g, coef, p + 1);
        const double dx = z10 - z00, dy = z01 - z00;
        acc += tv_norm(dx * dx + dy * dy);
    }
    return acc;
}

// the same for up to SUP_TRIAL_BATCH candidate steps at once: x and g are read once, every candidate's terms are
// accumulated in the order tv2d_share uses, so each result equals the one-at-a-time value bit for bit
template <typename T, int B>
__device__ void tv2d_share_batch(const PArgs<T>& A, const double* coef, double* acc) {
    const int64_t h = A.ny - 1, w = A.nx - 1;
    const int64_t total = h > 0 && w > 0 ? h * w : 0;
#pragma unroll
    for (int b = 0; b < B; ++b) acc[b] = 0.0;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < total; q += int64_t(gridDim.x) * blockDim.x) {
        const int64_t i = q / w, j = q - i * w;
        const int64_t p = i * A.nx + j;
        const double x00 = double(__ldcg(A.x + p)), x10 = double(__ldcg(A.x + p + A.nx)), x01 = double(__ldcg(A.x + p + 1));
        const double g00 = double(__ldcg(A.g + p)), g10 = double(__ldcg(A.g + p + A.nx)), g01 = double(__ldcg(A.g + p + 1));
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const double c = coef[b];
            const double z00 = c == 0.0 ? x00 : double(T(fma(-c, g00, x00)));
            const double z10 = c == 0.0 ? x10 : double(T(fma(-c, g10, x10)));
            const double z01 = c == 0.0 ? x01 : double(T(fma(-c, g01, x01)));
            const double dx = z10 - z00, dy = z01 - z00;
            acc[b] += tv_norm(dx * dx + dy * dy);
        }
    }
}

// TV3D value for B candidate steps at once (terms for i < nz-1, j < ny-1, k < nx-1; A-27)
template <typename T, int B>
__device__ void tv3d_share_batch(const PArgs<T>& A, const double* coef, double* acc) {
    const int64_t d = A.nz - 1, h = A.ny - 1, w = A.nx - 1;
    const int64_t total = d > 0 && h > 0 && w > 0 ? d * h * w : 0;
    const int64_t sz = A.ny * A.nx;
#pragma unroll
    for (int b = 0; b < B; ++b) acc[b] = 0.0;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < total; q += int64_t(gridDim.x) * blockDim.x) {
        const int64_t i = q / (h * w), r2 = q - i * h * w, j = r2 / w, k = r2 - j * w;
        const int64_t p = (i * A.ny + j) * A.nx + k;
        const double x0 = double(__ldcg(A.x + p)), xz = double(__ldcg(A.x + p + sz)), xy = double(__ldcg(A.x + p + A.nx)), xx = double(__ldcg(A.x + p + 1));
        double g0 = 0.0, gz = 0.0, gy = 0.0, gx = 0.0;
        bool any = false;
#pragma unroll
        for (int b = 0; b < B; ++b) any = any || coef[b] != 0.0;
        if (any) {
            g0 = double(__ldcg(A.g + p));
            gz = double(__ldcg(A.g + p + sz));
            gy = double(__ldcg(A.g + p + A.nx));
            gx = double(__ldcg(A.g + p + 1));
        }
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const double c = coef[b];
            const double z0 = c == 0.0 ? x0 : double(T(fma(-c, g0, x0)));
            const double zz = c == 0.0 ? xz : double(T(fma(-c, gz, xz)));
            const double zy = c == 0.0 ? xy : double(T(fma(-c, gy, xy)));
            const double zx = c == 0.0 ? xx : double(T(fma(-c, gx, xx)));
            const double dz = zz - z0, dy = zy - z0, dx = zx - z0;
            acc[b] += tv_norm((dz * dz + dy * dy) + dx * dx);
        }
    }
}

template <typename T, int B>
__device__ void tv1d_share_batch(const PArgs<T>& A, const double* coef, double* acc) {
#pragma unroll
    for (int b = 0; b < B; ++b) acc[b] = 0.0;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q + 1 < A.n; q += int64_t(gridDim.x) * blockDim.x) {
        const double x0 = double(__ldcg(A.x + q)), x1 = double(__ldcg(A.x + q + 1));
        const double g0 = double(__ldcg(A.g + q)), g1 = double(__ldcg(A.g + q + 1));
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const double c = coef[b];
            const double z0 = c == 0.0 ? x0 : double(T(fma(-c, g0, x0)));
            const double z1 = c == 0.0 ? x1 : double(T(fma(-c, g1, x1)));
            acc[b] += fabs(z1 - z0);
        }
    }
}

template <typename T>
__device__ double tv1d_share(const PArgs<T>& A, double coef) {
    double acc = 0.0;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q + 1 < A.n; q += int64_t(gridDim.x) * blockDim.x)
        acc += fabs(zval(A.x, A.g, coef, q + 1) - zval(A.x, A.g, coef, q));
    return acc;
}

// group-of-G row dot against z (dose) or against a plain vector
template <typename T, bool ZV>
__device__ __forceinline__ T coop_row_dot(const T* __restrict__ val, const int32_t* __restrict__ col, int64_t s, int64_t e,
                                          const T* __restrict__ x, const T* __restrict__ g, double coef, int gl, int G) {
    T a0 = T(0), a1 = T(0);
    int64_t k = s + gl;
    for (; k + G < e; k += 2 * int64_t(G)) {
        const int c0 = __ldcs(col + k), c1 = __ldcs(col + k + G);
        const T v0 = __ldcs(val + k), v1 = __ldcs(val + k + G);
        a0 += v0 * (ZV ? T(zval(x, g, coef, c0)) : __ldcg(x + c0));
        a1 += v1 * (ZV ? T(zval(x, g, coef, c1)) : __ldcg(x + c1));
    }
    if (k < e) a0 += __ldcs(val + k) * (ZV ? T(zval(x, g, coef, __ldcs(col + k))) : __ldcg(x + __ldcs(col + k)));
    T acc = a0 + a1;
    for (int o = G >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o, G);
    return acc;
}

template <typename T>
__device__ double dose_share(const PArgs<T>& A, double coef, bool store_r) {
    // f(z) = sum_i (D z)_i^2; optionally stores r = D z (used by the gradient with coef = 0)
    const int G = A.g_d;
    const int gl = threadIdx.x % G, lane = threadIdx.x & 31;
    const int64_t gid = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) / G;
    const int64_t ngroups = (int64_t(gridDim.x) * blockDim.x) / G;
    double acc = 0.0;
    for (int64_t i0 = gid - lane / G; i0 < A.md; i0 += ngroups) {  // warp-uniform bound
        const int64_t i = i0 + lane / G;
        const bool valid = i < A.md;
        const int64_t s = valid ? A.d_rowptr[i] : 0, e = valid ? A.d_rowptr[i + 1] : 0;
        const T r = coop_row_dot<T, true>(A.d_val, A.d_col, s, e, A.x, A.g, coef, gl, G);
        if (valid && gl == 0) {
            acc += double(r) * double(r);
            if (store_r) A.r[i] = r;
        }
    }
    return acc;
}

template <typename T, int OBJ>
__device__ __forceinline__ double objective_share(const PArgs<T>& A, double coef) {
    if (OBJ == SUP_OBJ_TV2D) return tv2d_share(A, coef);
    if (OBJ == SUP_OBJ_TV1D) return tv1d_share(A, coef);
    if (OBJ == SUP_OBJ_DOSE) return dose_share(A, coef, false);
    if (OBJ == SUP_OBJ_TV3D) {
        double acc[1];
        tv3d_share_batch<T, 1>(A, &coef, acc);
        return acc[0];
    }
    return 0.0;
}

// ---- TV passes over tiles: B candidate coefficients at once; z_b = round_T(x - c_b g) (c_b = 0: x itself) is formed on the fly
// from the tile's x and g.  Returns this thread's share F[b] of f(z_b) for every candidate and, when GRAD (B = 1), writes z
// to xo (if c != 0) and grad f(z) to go and returns the share S of sum (grad f(z))^2 (a term with t = 0 contributes 0, A-9).
// The value-only pass and the gradient pass assign pixels to threads and add terms in the SAME order, so f of a given z
// is the same bit pattern whichever pass computed it -- an accept test f(z) <= f(x) with z == x (a step below the storage
// type's resolution) must see equality.
__device__ __forceinline__ double tv_d2(double dx, double dy) { return fma(dx, dx, dy * dy); }
__device__ __forceinline__ double tv_d3(double dz, double dy, double dx) { return fma(dx, dx, fma(dy, dy, dz * dz)); }
template <typename T>
__device__ __forceinline__ double zform(double xv, double gv, double c) { return c == 0.0 ? xv : double(T(fma(-c, gv, xv))); }

// TV2D (A-8): g_ij = -(dx_ij+dy_ij)/t_ij [i<ny-1, j<nx-1] + dx_{i-1,j}/t_{i-1,j} [i>=1, j<nx-1] + dy_{i,j-1}/t_{i,j-1} [j>=1, i<ny-1].
// One CTA stages a TILE_H x TILE_W tile of x and of g plus a one-pixel halo in shared memory.
template <typename T, int B, bool GRAD>
__device__ void tv2d_pass(const PArgs<T>& A, const double* coef, T* __restrict__ xo, T* __restrict__ go, double* F, double& S, double* sm) {
    typedef double Tile2[TILE_W + 2 + 1];
    Tile2* tx = reinterpret_cast<Tile2*>(sm);
    Tile2* tg = reinterpret_cast<Tile2*>(sm + (TILE_H + 2) * (TILE_W + 2 + 1));
    const int64_t ny = A.ny, nx = A.nx;
    const int64_t tiles_y = (ny + TILE_H - 1) / TILE_H, tiles_x = (nx + TILE_W - 1) / TILE_W;
    bool any = false;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        F[b] = 0.0;
        any = any || coef[b] != 0.0;
    }
    double acc = 0.0;
    for (int64_t t = blockIdx.x; t < tiles_y * tiles_x; t += gridDim.x) {
        const int64_t ty = int64_t(unsigned(t) / unsigned(tiles_x)), txi = t - ty * tiles_x;  // (n < 2^31: a 32-bit division, a fifth of the 64-bit one)
        const int64_t i0 = ty * TILE_H - 1, j0 = txi * TILE_W - 1;  // top-left of the halo
        __syncthreads();
        for (int q = threadIdx.x; q < (TILE_H + 2) * (TILE_W + 2); q += SUP_THREADS) {
            const int li = q / (TILE_W + 2), lj = q - li * (TILE_W + 2);
            const int64_t i = i0 + li, j = j0 + lj;
            const bool in = i >= 0 && i < ny && j >= 0 && j < nx;
            const double xv = in ? double(__ldcg(A.x + i * nx + j)) : 0.0;
            const double gv = in && any ? double(__ldcg(A.g + i * nx + j)) : 0.0;
            if (B == 1) {
                tx[li][lj] = zform<T>(xv, gv, coef[0]);  // one candidate: the tile holds z itself
            } else {
                tx[li][lj] = xv;
                tg[li][lj] = gv;
            }
        }
        __syncthreads();
        for (int q = threadIdx.x; q < TILE_H * TILE_W; q += SUP_THREADS) {
            const int li = q / TILE_W + 1, lj = q % TILE_W + 1;
            const int64_t i = i0 + li, j = j0 + lj;
            if (i >= ny || j >= nx) continue;
            const bool own = i + 1 < ny && j + 1 < nx;
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const double cb = coef[b];
                auto Z = [&](int a, int bq) { return B == 1 ? tx[a][bq] : zform<T>(tx[a][bq], tg[a][bq], cb); };
                const double c = Z(li, lj);
                double gv = 0.0;
                if (own) {  // own term (i, j)
                    const double dx = Z(li + 1, lj) - c, dy = Z(li, lj + 1) - c;
                    const double d2 = tv_d2(dx, dy);
                    if (d2 > 0.0) {
                        const double ri = rsqrt(d2);
                        gv -= (dx + dy) * ri;
                        F[b] += d2 * ri;
                    }
                }
                if (GRAD) {
                    if (i >= 1 && j + 1 < nx) {  // term (i-1, j): dx_{i-1,j} = X_ij - X_{i-1,j}
                        const double bb = Z(li - 1, lj);
                        const double dx = c - bb, dy = Z(li - 1, lj + 1) - bb;
                        const double d2 = tv_d2(dx, dy);
                        if (d2 > 0.0) gv += dx * rsqrt(d2);
                    }
                    if (j >= 1 && i + 1 < ny) {  // term (i, j-1): dy_{i,j-1} = X_ij - X_{i,j-1}
                        const double bb = Z(li, lj - 1);
                        const double dx = Z(li + 1, lj - 1) - bb, dy = c - bb;
                        const double d2 = tv_d2(dx, dy);
                        if (d2 > 0.0) gv += dy * rsqrt(d2);
                    }
                    const T gs = T(gv);
                    go[i * nx + j] = gs;
                    if (cb != 0.0) xo[i * nx + j] = T(c);  // c is z rounded to T already
                    acc += double(gs) * double(gs);
                }
            }
        }
    }
    S = acc;
}

// TV3D (A-27): Eq. 15 with a third difference on an nz x ny x nx volume; a voxel receives +dz/t of term (i-1,j,k), +dy/t of
// (i,j-1,k), +dx/t of (i,j,k-1) and -(dz+dy+dx)/t of its own term.  Tile of TZ3 x TY3 x TX3 voxels plus a one-voxel halo.
#define TZ3 4
#define TY3 8
#define TX3 32
template <typename T, int B, bool GRAD>
__device__ void tv3d_pass(const PArgs<T>& A, const double* coef, T* __restrict__ xo, T* __restrict__ go, double* F, double& S, double* sm) {
    typedef double Vol3[TY3 + 2][TX3 + 2 + 1];
    Vol3* vx = reinterpret_cast<Vol3*>(sm);
    Vol3* vg = reinterpret_cast<Vol3*>(sm + (TZ3 + 2) * (TY3 + 2) * (TX3 + 2 + 1));
    const int64_t nz = A.nz, ny = A.ny, nx = A.nx;
    const int64_t tz = (nz + TZ3 - 1) / TZ3, ty = (ny + TY3 - 1) / TY3, txn = (nx + TX3 - 1) / TX3;
    bool any = false;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        F[b] = 0.0;
        any = any || coef[b] != 0.0;
    }
    double acc = 0.0;
    for (int64_t t = blockIdx.x; t < tz * ty * txn; t += gridDim.x) {
        const int64_t bz = int64_t(unsigned(t) / unsigned(ty * txn)), rem = t - bz * ty * txn, by = int64_t(unsigned(rem) / unsigned(txn)), bx = rem - by * txn;
        const int64_t i0 = bz * TZ3 - 1, j0 = by * TY3 - 1, k0 = bx * TX3 - 1;
        __syncthreads();
        for (int q = threadIdx.x; q < (TZ3 + 2) * (TY3 + 2) * (TX3 + 2); q += SUP_THREADS) {
            const int li = q / ((TY3 + 2) * (TX3 + 2)), r2 = q - li * (TY3 + 2) * (TX3 + 2), lj = r2 / (TX3 + 2), lk = r2 - lj * (TX3 + 2);
            const int64_t i = i0 + li, j = j0 + lj, k = k0 + lk;
            const bool in = i >= 0 && i < nz && j >= 0 && j < ny && k >= 0 && k < nx;
            const int64_t p = (i * ny + j) * nx + k;
            const double xv = in ? double(__ldcg(A.x + p)) : 0.0;
            const double gv = in && any ? double(__ldcg(A.g + p)) : 0.0;
            if (B == 1) {
                vx[li][lj][lk] = zform<T>(xv, gv, coef[0]);
            } else {
                vx[li][lj][lk] = xv;
                vg[li][lj][lk] = gv;
            }
        }
        __syncthreads();
        for (int q = threadIdx.x; q < TZ3 * TY3 * TX3; q += SUP_THREADS) {
            const int li = q / (TY3 * TX3) + 1, r2 = q % (TY3 * TX3), lj = r2 / TX3 + 1, lk = r2 % TX3 + 1;
            const int64_t i = i0 + li, j = j0 + lj, k = k0 + lk;
            if (i >= nz || j >= ny || k >= nx) continue;
            const bool own = i + 1 < nz && j + 1 < ny && k + 1 < nx;
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const double cb = coef[b];
                auto Z = [&](int a, int bq, int cq) { return B == 1 ? vx[a][bq][cq] : zform<T>(vx[a][bq][cq], vg[a][bq][cq], cb); };
                const double c = Z(li, lj, lk);
                double gv = 0.0;
                if (GRAD) {
                    if (i >= 1 && j + 1 < ny && k + 1 < nx) {  // term (i-1, j, k)
                        const double bb = Z(li - 1, lj, lk);
                        const double dz = c - bb, dy = Z(li - 1, lj + 1, lk) - bb, dx = Z(li - 1, lj, lk + 1) - bb;
                        const double d2 = tv_d3(dz, dy, dx);
                        if (d2 > 0.0) gv += dz * rsqrt(d2);
                    }
                    if (j >= 1 && i + 1 < nz && k + 1 < nx) {  // term (i, j-1, k)
                        const double bb = Z(li, lj - 1, lk);
                        const double dz = Z(li + 1, lj - 1, lk) - bb, dy = c - bb, dx = Z(li, lj - 1, lk + 1) - bb;
                        const double d2 = tv_d3(dz, dy, dx);
                        if (d2 > 0.0) gv += dy * rsqrt(d2);
                    }
                    if (k >= 1 && i + 1 < nz && j + 1 < ny) {  // term (i, j, k-1)
                        const double bb = Z(li, lj, lk - 1);
                        const double dz = Z(li + 1, lj, lk - 1) - bb, dy = Z(li, lj + 1, lk - 1) - bb, dx = c - bb;
                        const double d2 = tv_d3(dz, dy, dx);
                        if (d2 > 0.0) gv += dx * rsqrt(d2);
                    }
                }
                if (own) {
                    const double dz = Z(li + 1, lj, lk) - c, dy = Z(li, lj + 1, lk) - c, dx = Z(li, lj, lk + 1) - c;
                    const double d2 = tv_d3(dz, dy, dx);
                    if (d2 > 0.0) {
                        const double ri = rsqrt(d2);
                        gv -= ((dz + dy) + dx) * ri;
                        F[b] += d2 * ri;
                    }
                }
                if (GRAD) {
                    const T gs = T(gv);
                    const int64_t p = (i * ny + j) * nx + k;
                    go[p] = gs;
                    if (cb != 0.0) xo[p] = T(c);
                    acc += double(gs) * double(gs);
                }
            }
        }
    }
    S = acc;
}

// TV1D (A-16), same contract; the value-only pass walks the same elements in the same order
template <typename T, int B, bool GRAD>
__device__ void tv1d_pass(const PArgs<T>& A, const double* coef, T* __restrict__ xo, T* __restrict__ go, double* F, double& S, double*) {
    bool any = false;
#pragma unroll
    for (int b = 0; b < B; ++b) {
        F[b] = 0.0;
        any = any || coef[b] != 0.0;
    }
    double acc = 0.0;
    for (int64_t q = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q < A.n; q += int64_t(gridDim.x) * blockDim.x) {
        const double x0 = double(__ldcg(A.x + q)), xl = q >= 1 ? double(__ldcg(A.x + q - 1)) : 0.0, xr = q + 1 < A.n ? double(__ldcg(A.x + q + 1)) : 0.0;
        double g0 = 0.0, gl = 0.0, gr = 0.0;
        if (any) {
            g0 = double(__ldcg(A.g + q));
            gl = q >= 1 ? double(__ldcg(A.g + q - 1)) : 0.0;
            gr = q + 1 < A.n ? double(__ldcg(A.g + q + 1)) : 0.0;
        }
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const double cb = coef[b];
            const double c = zform<T>(x0, g0, cb);
            double gv = 0.0;
            if (GRAD && q >= 1) {
                const double dl = c - zform<T>(xl, gl, cb);
                gv += double((dl > 0.0) - (dl < 0.0));
            }
            if (q + 1 < A.n) {
                const double dr = zform<T>(xr, gr, cb) - c;
                gv -= double((dr > 0.0) - (dr < 0.0));
                F[b] += fabs(dr);
            }
            if (GRAD) {
                go[q] = T(gv);
                if (cb != 0.0) xo[q] = T(c);
                acc += gv * gv;
            }
        }
    }
    S = acc;
}

// ---- the perturbation phase, TV objectives ---------------------------------------------------------------------
// Buffers: (xc, gc) hold the current inner iterate x^{k,n} and its gradient, (xo, go) receive the candidate z and its gradient
// (a tile's halo needs the neighbours' x and g, so a pass cannot work in place); on acceptance the pairs swap.
template <typename T, int OBJ>
__device__ __forceinline__ void tv_gz(const PArgs<T>& V, double c, T* xo, T* go, double& F, double& S, double* sm) {
    if (OBJ == SUP_OBJ_TV2D) tv2d_pass<T, 1, true>(V, &c, xo, go, &F, S, sm);
    else if (OBJ == SUP_OBJ_TV3D) tv3d_pass<T, 1, true>(V, &c, xo, go, &F, S, sm);
    else tv1d_pass<T, 1, true>(V, &c, xo, go, &F, S, sm);
}
// doubles of shared memory the tile passes of an objective need (x tile + g tile)
template <int OBJ>
__host__ __device__ constexpr int tv_tile_doubles() {
    return OBJ == SUP_OBJ_TV2D ? 2 * (TILE_H + 2) * (TILE_W + 2 + 1) : (OBJ == SUP_OBJ_TV3D ? 2 * (TZ3 + 2) * (TY3 + 2) * (TX3 + 2 + 1) : 1);
}
template <typename T, int OBJ, int B>
__device__ __forceinline__ void tv_share_batch(const PArgs<T>& V, const double* coef, double* acc, double* sm) {
    double unused;
    if (OBJ == SUP_OBJ_TV2D) tv2d_pass<T, B, false>(V, coef, nullptr, nullptr, acc, unused, sm);
    else if (OBJ == SUP_OBJ_TV3D) tv3d_pass<T, B, false>(V, coef, nullptr, nullptr, acc, unused, sm);
    else tv1d_pass<T, B, false>(V, coef, nullptr, nullptr, acc, unused, sm);
}

template <typename T, int OBJ>
__global__ void __launch_bounds__(SUP_THREADS) k_perturb_tv(PArgs<T> Ain) {
    const PArgs<T>& A = Ain;
    if (*(volatile int*)&Ain.st->stop) return;  // the stopping rule fired earlier in this run: every CTA sees the same flag
    __shared__ double tile_mem[tv_tile_doubles<OBJ>()];
    T* xc = Ain.x;
    T* gc = Ain.g;
    T* xo = Ain.x2;
    T* go = Ain.g2;
    auto view = [&]() {  // the argument block with the current buffers
        PArgs<T> V = Ain;
        V.x = xc;
        V.g = gc;
        return V;
    };
    DevState* st = A.st;
    long long ell = *(volatile long long*)&st->ell;
    double apow = *(volatile double*)&st->apow;  // a^ell, running product (A-20)
    const long long k = *(volatile long long*)&st->k;
    long long ndec = *(volatile long long*)&st->n_dec;
    GridBar gen = {*(volatile unsigned long long*)&st->bar_base, 0u};  // read before this CTA's first arrival (CTA 0 rewrites it at the end)
    // Eq. 11's reference: like every other field of the state it is read HERE, before this CTA's first arrival at a grid barrier --
    // CTA 0 rewrites it at the end of the kernel, which it can only reach after every CTA has arrived at the first barrier
    const double f_ref = *(volatile double*)&st->f_ref;
    long long trials = 0;
    // restarted perturbations (A-24): at the start of sweep k = r * n_restart the exponent is reset to r
    if (A.n_restart > 0 && k > 0 && k % A.n_restart == 0) {
        ell = k / A.n_restart;
        apow = 1.0;
        for (long long q = 0; q < ell; ++q) apow *= A.a;
    }
    int warn = 0, fault = 0;
    double pend = 0.0;  // step accepted in the last reduction step and not yet written anywhere: x^{k,N} = xc - pend gc
    double* P = A.partials;
    constexpr int B = SUP_TRIAL_BATCH;
    constexpr int PSTRIDE = SUP_MAX_PARTIALS / B;  // partial slots per reduced value (two buffers of SUP_MAX_PARTIALS: barrier parity)
    bool ok = true;

    auto log_trial = [&](double fz, double fxv, bool acc) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            if (A.decisions && ndec < A.cap) A.decisions[ndec] = acc ? 1 : 0;
            if (A.decision_f && ndec < A.cap) {
                A.decision_f[2 * ndec] = fz;
                A.decision_f[2 * ndec + 1] = fxv;
            }
        }
        ++ndec;
    };
    auto step_coef = [&](double s, long long jloc, double* coef, int cnt) {
        // a^(exponent of candidate 0) by successive multiplication from 1, like the oracle (A-20): PER_TRIAL carries the
        // running product a^l across trials and sweeps; PER_SWEEP rebuilds a^(k+j) (k is small)
        double ap = apow;
        if (A.policy != SUP_STEP_PER_TRIAL) {
            ap = 1.0;
            for (long long q = 0; q < k + jloc; ++q) ap *= A.a;
        }
        for (int b = 0; b < cnt; ++b) {
            coef[b] = s > 0.0 ? (A.beta0 * ap) / s : 0.0;
            ap *= A.a;
        }
    };

    // pass 0: gradient of x^{k,0}; f(x^{k,0}) and ||g||^2 come with it
    double fx, s;
    {
        double v[2];
        tv_gz<T, OBJ>(view(), 0.0, xo, gc, v[0], v[1], tile_mem);
        ok = grid_reduce<2>(st, P, PSTRIDE, v, gen);
        fx = v[0];
        s = sqrt(v[1]);
        if (!isfinite(fx)) fault |= 2;
    }
    // Eq. 11 (A-30): beta = (f - f_ref)/||g|| when f > f_ref, else 0; the step x - ((f - f_ref)/||g||^2) g is
    // taken as it is -- no trial loop, no exponent.  Same passes as an always-accepted first candidate: 1 + N in all.
    const bool adaptive = A.step_rule == SUP_RULE_ADAPTIVE;
    const double f_start = fx;
    for (int nred = 0; ok && adaptive && nred < A.N; ++nred) {
        const bool take = fx > f_ref && s > 0.0;
        log_trial(f_ref, fx, take);
        if (!take) continue;  // beta = 0: x^{k,n+1} = x^{k,n}, and so for every later step of this phase
        ++trials;
        const double c = ((fx - f_ref) / s) / s;
        if (nred == A.N - 1) {
            pend = c;  // applied by the final write below; f of the final point is not evaluated
            break;
        }
        double v[2];
        tv_gz<T, OBJ>(view(), c, xo, go, v[0], v[1], tile_mem);
        ok = grid_reduce<2>(st, P, PSTRIDE, v, gen);
        if (!ok) break;
        fx = v[0];
        s = sqrt(v[1]);
        if (!isfinite(fx)) fault |= 2;
        T* t = gc;
        gc = go;
        go = t;
        if (c != 0.0) {
            t = xc;
            xc = xo;
            xo = t;
        }
    }
    for (int nred = 0; ok && !adaptive && nred < A.N; ++nred) {
        const bool last = nred == A.N - 1;
        bool accepted = false;
        long long jloc = 0;
        int trial = 0;
        if (!last) {
            // First candidate, evaluated completely: z, f(z), grad f(z), ||grad f(z)||^2 in one pass.  Accepted (the common
            // case once beta is small), the next reduction step starts from (xo, go) without another pass.
            double c0;
            step_coef(s, jloc, &c0, 1);
            double v[2];
            tv_gz<T, OBJ>(view(), c0, xo, go, v[0], v[1], tile_mem);
            ok = grid_reduce<2>(st, P, PSTRIDE, v, gen);
            if (!ok) break;
            const bool acc = v[0] <= fx;  // NaN compares false -> rejected (A-11)
            ++ell;
            apow *= A.a;
            ++jloc;
            ++trials;
            ++trial;
            log_trial(v[0], fx, acc);
            if (acc) {
                accepted = true;
                fx = v[0];
                s = sqrt(v[1]);
                T* t = gc;
                gc = go;
                go = t;
                if (c0 != 0.0) {
                    t = xc;
                    xc = xo;
                    xo = t;
                }
            }
        }
        // Otherwise (or in the last reduction step, whose gradient nobody needs): the next B candidates per pass, values only,
        // decided strictly in order -- the first with f(z) <= f(x^{k,n}) is accepted, later ones are discarded uncounted.
        double cf = 0.0;
        while (ok && !accepted && trial < SUP_J_MAX) {
            double coef[B], fzb[B];
            // The first candidate of the LAST step goes alone (in the steady state it is accepted: evaluating B candidates for it
            // was 8 times the arithmetic, ~15 us per sweep at 512 x 512); after a rejection B at a time.  Same bits either way.
            const int nb = trial == 0 ? 1 : B;
            step_coef(s, jloc, coef, nb);
            if (nb == 1) {
                tv_share_batch<T, OBJ, 1>(view(), coef, fzb, tile_mem);
                ok = grid_reduce<1>(st, P, PSTRIDE, fzb, gen);
            } else {
                tv_share_batch<T, OBJ, B>(view(), coef, fzb, tile_mem);
                ok = grid_reduce<B>(st, P, PSTRIDE, fzb, gen);
            }
            if (!ok) break;
            for (int b = 0; b < nb && !accepted && trial < SUP_J_MAX; ++b) {
                const bool acc = fzb[b] <= fx;
                ++ell;
                apow *= A.a;
                ++jloc;
                ++trials;
                ++trial;
                log_trial(fzb[b], fx, acc);
                if (acc) {
                    accepted = true;
                    cf = coef[b];
                    fx = fzb[b];
                }
            }
            if (accepted) {
                if (last) {
                    pend = cf;  // applied by the final write below
                } else {
                    // the gradient at the accepted z (f(z) again, in this pass's summation order, carried from here on)
                    double v[2];
                    tv_gz<T, OBJ>(view(), cf, xo, go, v[0], v[1], tile_mem);
                    ok = grid_reduce<2>(st, P, PSTRIDE, v, gen);
                    if (!ok) break;
                    fx = v[0];
                    s = sqrt(v[1]);
                    T* t = gc;
                    gc = go;
                    go = t;
                    if (cf != 0.0) {
                        t = xc;
                        xc = xo;
                        xo = t;
                    }
                }
            }
        }
        if (ok && !accepted) warn |= 1;  // A-12: step skipped
    }
    // leave the final iterate in the caller's x and in the gather mirror (element-wise: no barrier needed)
    if (ok && (pend != 0.0 || xc != Ain.x || A.xg)) {
        // four elements per thread and trip, their loads issued before the first store (one L2 round trip per trip instead of four)
        const int64_t nth = int64_t(gridDim.x) * blockDim.x;
        for (int64_t q0 = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; q0 < A.n; q0 += 4 * nth) {
            T v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int64_t q = q0 + u * nth;
                v[u] = q < A.n ? T(zval(xc, gc, pend, q)) : T(0);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int64_t q = q0 + u * nth;
                if (q >= A.n) break;
                if (pend != 0.0 || xc != Ain.x) Ain.x[q] = v[u];
                if (A.xg) A.xg[sup_gmap(A.xmap, int(q))] = v[u];
            }
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        st->ell = ell;
        st->apow = apow;
        st->n_dec = ndec;
        st->n_trials += trials;
        st->sweep_trials += trials;
        st->f = fx;
        if (ok) st->bar_base = gen.target;  // where the next launch's barriers start
        if (adaptive && f_start <= f_ref) st->f_ref = A.shrink * f_start;  // the reference was reached: move it below (A-30)
        if (warn) atomicOr(&st->warn, warn);
        if (fault) atomicOr(&st->fault, fault);
    }
}

// ---- stand-alone objective value (sup_objective, trace mode) -------------------------------------------------
template <typename T, int OBJ>
__global__ void __launch_bounds__(SUP_THREADS) k_objective(PArgs<T> A) {
    const double sh = cta_sum(objective_share<T, OBJ>(A, 0.0));
    if (threadIdx.x == 0) A.partials[blockIdx.x] = sh;
}
__global__ void k_sum_final(const double* __restrict__ partials, int np, double* __restrict__ out) {
    __shared__ double shm[SUP_THREADS];
    double s = 0.0;
    for (int q = threadIdx.x; q < np; q += SUP_THREADS) s += partials[q];
    shm[threadIdx.x] = s;
    __syncthreads();
    for (int o = SUP_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) shm[threadIdx.x] += shm[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = shm[0];
}

// ---- host side --------------------------------------------------------------------------------------------------

template <typename T>
static const void* perturb_kernel(int objective) {
    switch (objective) {
        case SUP_OBJ_TV2D: return reinterpret_cast<const void*>(&k_perturb_tv<T, SUP_OBJ_TV2D>);
        case SUP_OBJ_TV1D: return reinterpret_cast<const void*>(&k_perturb_tv<T, SUP_OBJ_TV1D>);
        case SUP_OBJ_TV3D: return reinterpret_cast<const void*>(&k_perturb_tv<T, SUP_OBJ_TV3D>);
    }
    return nullptr;
}

// grid of the cooperative kernel: enough CTAs for the work, never more than can be co-resident or than the
// partial-sum slots; small problems get small grids (a barrier costs more with more CTAs)
int sup_perturb_grid(sup_ctx* h, int objective) {
    const void* fn = h->dt == SUP_F32 ? perturb_kernel<float>(objective) : perturb_kernel<double>(objective);
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, SUP_THREADS, 0) != cudaSuccess || per_sm < 1) return 0;
    int64_t cap = int64_t(per_sm) * h->num_sms;
    if (cap > SUP_MAX_PARTIALS) cap = SUP_MAX_PARTIALS;
    int64_t want;
    if (objective == SUP_OBJ_DOSE) {
        want = (h->D.rows * h->g_d + SUP_THREADS - 1) / SUP_THREADS;
        if (want > 4 * int64_t(h->num_sms)) want = 4 * int64_t(h->num_sms);
    } else {
        want = (h->n + 4 * SUP_THREADS - 1) / (4 * SUP_THREADS);  // about four elements per thread
        if (want > 2 * int64_t(h->num_sms)) want = 2 * int64_t(h->num_sms);
        if (want > SUP_MAX_PARTIALS / SUP_TRIAL_BATCH) want = SUP_MAX_PARTIALS / SUP_TRIAL_BATCH;  // one partial row per candidate
    }
    if (want < 1) want = 1;
    return int(want < cap ? want : cap);
}

sup_status sup_launch_perturb(sup_ctx* h, void* x, const PerturbParams& pp) {
    if (pp.objective == SUP_OBJ_MEAN) return sup_launch_perturb_mean(h, x, pp);
    if (pp.objective == SUP_OBJ_DOSE) {
        if (h->gram && h->dose_mode == 0) return sup_launch_perturb_dose_gram(h, x, pp);
        if (!(h->D.plan.ok && h->DT.plan.ok)) return sup_fail(h, SUP_ERR_STATE, "the dose perturbation runs on the staged product kernels (sup_set_row_mode)");
        return sup_launch_perturb_dose_staged(h, x, pp);
    }
    if (sup_perturb_small_eligible(h, pp)) return sup_launch_perturb_small(h, x, pp);  // small images: one cluster (sup_perturb_small.cu)
    const int grid = sup_perturb_grid(h, pp.objective);
    if (grid < 1) return sup_fail(h, SUP_ERR_CUDA, "perturbation kernel cannot be made resident");
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(unsigned(grid));
    cfg.blockDim = dim3(SUP_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (h->dt == SUP_F32) {
        PArgs<float> A = sup_make_perturb_args<float>(h, x, pp);
        void* args[] = {&A};
        SUP_CUDA(h, cudaLaunchKernelExC(&cfg, perturb_kernel<float>(pp.objective), args));
    } else {
        PArgs<double> A = sup_make_perturb_args<double>(h, x, pp);
        void* args[] = {&A};
        SUP_CUDA(h, cudaLaunchKernelExC(&cfg, perturb_kernel<double>(pp.objective), args));
    }
    h->launches++;
    return SUP_OK;
}

template <typename T>
static void launch_objective_t(sup_ctx* h, const void* x, int kind, int64_t nz, int64_t ny, int64_t nx, double* out_dev) {
    PerturbParams pp = {};
    pp.nz = nz;
    pp.objective = kind;
    pp.ny = ny;
    pp.nx = nx;
    PArgs<T> A = sup_make_perturb_args<T>(h, const_cast<void*>(x), pp);
    int grid = h->num_sms * 4;
    if (grid > SUP_MAX_PARTIALS) grid = SUP_MAX_PARTIALS;
    const int64_t work = kind == SUP_OBJ_DOSE ? h->D.rows * h->g_d : h->n;
    grid = sup_grid_for(work, SUP_THREADS, grid);
    if (kind == SUP_OBJ_TV2D) k_objective<T, SUP_OBJ_TV2D><<<grid, SUP_THREADS, 0, h->stream>>>(A);
    else if (kind == SUP_OBJ_TV3D) k_objective<T, SUP_OBJ_TV3D><<<grid, SUP_THREADS, 0, h->stream>>>(A);
    else if (kind == SUP_OBJ_TV1D) k_objective<T, SUP_OBJ_TV1D><<<grid, SUP_THREADS, 0, h->stream>>>(A);
    else if (kind == SUP_OBJ_DOSE) k_objective<T, SUP_OBJ_DOSE><<<grid, SUP_THREADS, 0, h->stream>>>(A);
    else k_objective<T, SUP_OBJ_NONE><<<1, SUP_THREADS, 0, h->stream>>>(A);
    k_sum_final<<<1, SUP_THREADS, 0, h->stream>>>(h->partials, kind == SUP_OBJ_NONE ? 1 : grid, out_dev);
    h->launches += 2;
}

void sup_launch_objective(sup_ctx* h, const void* x, int kind, int64_t nz, int64_t ny, int64_t nx, double* out_dev) {
    if (kind == SUP_OBJ_MEAN) {  // f_Mean(x) = <(1/N_S) D_S^T 1, x>
        const int np = sup_launch_mean_value(h, x);
        k_sum_final<<<1, SUP_THREADS, 0, h->stream>>>(h->partials, np, out_dev);
        h->launches++;
        return;
    }
    if (h->dt == SUP_F32) launch_objective_t<float>(h, x, kind, nz, ny, nx, out_dev);
    else launch_objective_t<double>(h, x, kind, nz, ny, nx, out_dev);
}

__global__ void k_begin_run(DevState* st, long long ell0, long long k0, double apow0, long long n_iter, double f_ref) {
    st->f_ref = f_ref;
    st->f_start = 0.0;
    st->n_iter = n_iter;
    st->n_done = 0;
    st->stop = 0;
    st->stop_reason = 0;
    st->consec = 0;
    st->prox_prev = st->f_prev = st->prox_cur = st->f_cur = 0.0;
    st->step = 0.0;
    st->cf = 0.0;
    st->ell = ell0;
    st->apow = apow0;
    st->k = k0;
    st->it = 0;
    st->n_trials = 0;
    st->sweep_trials = 0;
    st->n_dec = 0;
    st->warn = 0;
    st->fault = 0;
    st->bar_count = 0;
    st->bar_base = 0;
}
void sup_launch_begin_run(sup_ctx* h, int64_t ell0, int64_t k0, double a, int64_t n_iter, double f_ref) {
    // a^l0: exactly 1 for a fresh run, so the running product below reproduces the oracle's step sizes bit for bit (A-20)
    double apow0 = 1.0;
    for (int64_t i = 0; i < ell0; ++i) apow0 *= a;  // (ell0 is bounded by the argument check: the product stays exact-by-construction)
    k_begin_run<<<1, 1, 0, h->stream>>>(h->state, ell0, k0, apow0, n_iter, f_ref);
    h->launches++;
}
