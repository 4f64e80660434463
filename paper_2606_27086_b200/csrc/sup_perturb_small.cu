// sup_perturb_small.cu -- the TV2D perturbation phase (Algorithm 1 lines 4-17; Eq. 11 with SUP_RULE_ADAPTIVE) for
// SMALL images: ONE thread-block cluster instead of a grid with a software barrier.
//
// k_perturb_tv (sup_perturb.cu) spreads an image over up to 2 x 148 CTAs and pays a global-memory round trip per pass: the candidate
// z and its gradient go through L2, and every pass ends in a software grid barrier (~3 us).  For a 64 x 64 or 128 x 128 image
// (BASELINE.json configs[0] and [1]) that is all latency: 53 us for the 1 + N = 6 passes of config 1, three times its basic sweep.
// Here the image lives in the shared memory of a cluster of 8 CTAs (16 above 8 192 pixels: config 2's phase 69 -> 51 us) in contiguous row blocks, the current iterate x, its
// gradient g and the candidate z never leave the SMs during the phase, neighbouring rows of another CTA are read through
// distributed shared memory, the two sums of a pass (f(z) and ||grad f(z)||^2) are exchanged by DSMEM stores, and the only
// synchronisation is the hardware cluster barrier (two per pass).  Candidates are evaluated one at a time (there is no barrier
// cost to amortise over a batch), strictly in order: the trial / decision / l sequence is Algorithm 1's, as in k_perturb_tv.
// A pixel's terms are computed by the same thread with the same code whether or not the gradient is wanted, and the sums are
// taken in a fixed order, so f(z) is one bit pattern per z (an accept test with z == x sees equality).
//
// Eligible: TV2D, ny >= SMALL_C rows, at most SMALL_LOCAL_MAX pixels per CTA (n <= 32 768 for row counts that divide evenly).
// sup_set_perturb_mode(h, 1) keeps the grid kernel for such images (tests run both).
#include <cooperative_groups.h>

#include "sup_internal.cuh"
#include "sup_perturb_args.cuh"

namespace cg = cooperative_groups;

#define SMALL_THR 512
#define SMALL_C 8       // portable cluster size: images of up to 8 192 pixels
#define SMALL_CMAX 16   // non-portable size (opt-in, B200 has it): larger images, where a pass is bound by the fp64 work per CTA
#define SMALL_PPT 8
#define SMALL_LOCAL_MAX (SMALL_THR * SMALL_PPT)  // pixels one CTA holds
#define SMALL_NB 4        // candidates per value-only pass after a rejected first candidate

struct SmallShared {
    double ws[SMALL_THR / 32][SMALL_NB];  // per-warp partial sums of a reduction
    double part[2][SMALL_CMAX][SMALL_NB];    // [parity][rank][value]: the CTAs' sums, written by their owners into EVERY CTA's copy
};

// sums v[0..NV) over the whole cluster; on return every thread holds the totals.  Fixed order: lanes (shuffle tree), warps in index
// order, CTAs in rank order.  Contains one cluster barrier, after which nobody reads the array the terms were computed from.
template <int NV>
__device__ __forceinline__ void small_reduce(cg::cluster_group& cl, SmallShared& sh, unsigned& parity, double* v) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int b = 0; b < NV; ++b)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[b] += __shfl_xor_sync(0xffffffffu, v[b], o);
    if (lane == 0)
#pragma unroll
        for (int b = 0; b < NV; ++b) sh.ws[wid][b] = v[b];
    __syncthreads();
    const unsigned nb = cl.num_blocks(), me = cl.block_rank();
    if (threadIdx.x < NV * nb) {  // thread (b, r): this CTA's sum b into CTA r's copy
        const int b = threadIdx.x % NV;
        const unsigned r = threadIdx.x / NV;
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < SMALL_THR / 32; ++w) t += sh.ws[w][b];
        *cl.map_shared_rank(&sh.part[parity][me][b], r) = t;
    }
    cl.sync();
#pragma unroll
    for (int b = 0; b < NV; ++b) {
        double t = 0.0;
        for (unsigned r = 0; r < nb; ++r) t += sh.part[parity][r][b];
        v[b] = t;
    }
    parity ^= 1u;
}

// TV terms of the pixels this thread owns (A-8, as tv2d_pass of sup_perturb.cu): share F of f(z); with GRAD the gradient of the owned
// pixels into gout[] (rounded to T) and the share S of sum g^2.  zl: this CTA's rows [r0, r1) of z; zp / zn: the last row of the
// CTA before and the first row of the CTA after (distributed shared memory), valid where such a row exists.
template <typename T, bool GRAD, int PPT>
__device__ __forceinline__ void small_terms(const T* zl, const T* zp, const T* zn, int r0, int r1, int ny, int nx, double& F, double& S, T* gout,
                                            const int* pij) {
    F = 0.0;
    S = 0.0;
    const int nloc = (r1 - r0) * nx;
    auto row = [&](int i) -> const T* { return i < r0 ? zp : (i >= r1 ? zn : zl + (i - r0) * nx); };
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
        const int q = threadIdx.x + k * SMALL_THR;
        if (q >= nloc) break;
        const int il = pij[k] >> 16, j = pij[k] & 0xffff, i = r0 + il;  // (row, column) of the pixel: divided once, at the start of the kernel
        const T* ri = zl + il * nx;
        const double c = double(ri[j]);
        double gv = 0.0;
        if (i + 1 < ny && j + 1 < nx) {  // own term (i, j)
            const double dx = double(row(i + 1)[j]) - c, dy = double(ri[j + 1]) - c;
            const double d2 = fma(dx, dx, dy * dy);
            if (d2 > 0.0) {
                const double rs = rsqrt(d2);
                gv -= (dx + dy) * rs;
                F += d2 * rs;
            }
        }
        if (GRAD) {
            if (i >= 1 && j + 1 < nx) {  // term (i-1, j)
                const T* rm = row(i - 1);
                const double bb = double(rm[j]);
                const double dx = c - bb, dy = double(rm[j + 1]) - bb;
                const double d2 = fma(dx, dx, dy * dy);
                if (d2 > 0.0) gv += dx * rsqrt(d2);
            }
            if (j >= 1 && i + 1 < ny) {  // term (i, j-1)
                const double bb = double(ri[j - 1]);
                const double dx = double(row(i + 1)[j - 1]) - bb, dy = c - bb;
                const double d2 = fma(dx, dx, dy * dy);
                if (d2 > 0.0) gv += dy * rsqrt(d2);
            }
            const T gs = T(gv);
            gout[k] = gs;
            S += double(gs) * double(gs);
        }
    }
}

// f(z_b), z_b = round_T(x - c_b g), for SMALL_NB candidates at once, z formed on the fly from x and g (this CTA's rows and the first row
// of the CTA after it, read through distributed shared memory): the same operations on the same values as small_terms<T, false> on
// a stored z_b, hence the same bits.  No z array, no cluster barrier before the terms: one barrier (the reduction's) per SMALL_NB trials.
template <typename T>
__device__ __forceinline__ void small_terms_batch(const T* xl, const T* gl, const T* xn, const T* gn, int r0, int r1, int ny, int nx, const double* coef,
                                               double* F) {
#pragma unroll
    for (int b = 0; b < SMALL_NB; ++b) F[b] = 0.0;
    const int nloc = (r1 - r0) * nx;
#pragma unroll 1
    for (int q = threadIdx.x; q < nloc; q += SMALL_THR) {
        const int il = q / nx, j = q - il * nx, i = r0 + il;
        if (i + 1 >= ny || j + 1 >= nx) continue;
        const bool below_local = i + 1 < r1;
        const double x0 = double(xl[q]), g0 = double(gl[q]);
        const double x1 = double(below_local ? xl[q + nx] : xn[j]), g1 = double(below_local ? gl[q + nx] : gn[j]);
        const double x2 = double(xl[q + 1]), g2v = double(gl[q + 1]);
#pragma unroll
        for (int b = 0; b < SMALL_NB; ++b) {
            const double cb = coef[b];
            const double c = cb == 0.0 ? x0 : double(T(fma(-cb, g0, x0)));
            const double zd = cb == 0.0 ? x1 : double(T(fma(-cb, g1, x1)));
            const double zr = cb == 0.0 ? x2 : double(T(fma(-cb, g2v, x2)));
            const double dx = zd - c, dy = zr - c;
            const double d2 = fma(dx, dx, dy * dy);
            if (d2 > 0.0) F[b] += d2 * rsqrt(d2);
        }
    }
}

// PPT: pixels per thread the kernel is built for (2: images of up to 1 024 pixels per CTA -- configs 1 and 2 -- with a fraction of
// the registers and of the unrolled code of the general PPT = SMALL_PPT build)
template <typename T, int PPT>
__global__ void __launch_bounds__(SMALL_THR, 1) k_perturb_tv2d_small(PArgs<T> A, int rows_max) {
    cg::cluster_group cl = cg::this_cluster();
    DevState* st = A.st;
    if (*(volatile int*)&st->stop) return;  // every CTA sees the same flag (set by an earlier kernel of the run)
    sup_pdl_trigger();  // the forward product that follows may become resident on the idle SMs and fill its ring meanwhile
    extern __shared__ __align__(16) unsigned char small_raw[];
    __shared__ SmallShared sh;
    const int ny = int(A.ny), nx = int(A.nx);
    const unsigned me = cl.block_rank(), nb = cl.num_blocks();
    const int r0 = int(int64_t(me) * ny / nb), r1 = int(int64_t(me + 1) * ny / nb);  // >= 1 row each (ny >= nb)
    const int nloc = (r1 - r0) * nx;
    const int cap = rows_max * nx;
    T* sX = reinterpret_cast<T*>(small_raw);
    T* sG = sX + cap;
    T* sZ = sG + cap;
    // the neighbours' rows this CTA's terms touch: last row of the CTA before, first row of the CTA after
    const int rows_prev = me > 0 ? int(int64_t(me) * ny / nb) - int(int64_t(me - 1) * ny / nb) : 0;
    auto prev_last = [&](T* arr) -> const T* { return me > 0 ? cl.map_shared_rank(arr, me - 1) + (rows_prev - 1) * nx : arr; };
    auto next_first = [&](T* arr) -> const T* { return me + 1 < nb ? cl.map_shared_rank(arr, me + 1) : arr; };

    // run state: read before the first cluster barrier, written by CTA 0 at the very end
    long long ell = *(volatile long long*)&st->ell;
    double apow = *(volatile double*)&st->apow;
    const long long k = *(volatile long long*)&st->k;
    long long ndec = *(volatile long long*)&st->n_dec;
    const double f_ref = *(volatile double*)&st->f_ref;
    long long trials = 0;
    if (A.n_restart > 0 && k > 0 && k % A.n_restart == 0) {  // restarted perturbations (A-24)
        ell = k / A.n_restart;
        apow = 1.0;
        for (long long q = 0; q < ell; ++q) apow *= A.a;
    }
    int warn = 0, fault = 0;
    unsigned parity = 0;
    const int64_t g0 = int64_t(r0) * nx;  // first pixel of this CTA in the image
    for (int q = threadIdx.x; q < nloc; q += SMALL_THR) sX[q] = __ldcg(A.x + g0 + q);
    cl.sync();

    auto log_trial = [&](double fz, double fxv, bool acc) {
        if (me == 0 && threadIdx.x == 0) {
            if (A.decisions && ndec < A.cap) A.decisions[ndec] = acc ? 1 : 0;
            if (A.decision_f && ndec < A.cap) {
                A.decision_f[2 * ndec] = fz;
                A.decision_f[2 * ndec + 1] = fxv;
            }
        }
        ++ndec;
    };
    auto step_coef = [&](double s, long long jloc) {  // (beta0 a^exponent) / ||g||, exponent as the running product (A-20)
        double ap = apow;
        if (A.policy != SUP_STEP_PER_TRIAL) {
            ap = 1.0;
            for (long long q = 0; q < k + jloc; ++q) ap *= A.a;
        }
        return s > 0.0 ? (A.beta0 * ap) / s : 0.0;
    };
    T g2[PPT];
    int pij[PPT];  // (local row << 16) | column of the pixels this thread owns (rows and columns are <= 4096 here)
#pragma unroll
    for (int kk = 0; kk < PPT; ++kk) {
        const int q = threadIdx.x + kk * SMALL_THR;
        const int il = q < nloc ? q / nx : 0;
        pij[kk] = (il << 16) | (q < nloc ? q - il * nx : 0);
    }
    bool moved = false;  // x differs from what the caller passed in
    auto form_z = [&](double c) {  // z = round_T(x - c g) for the owned pixels (c = 0: x itself), then visible to the cluster
        for (int q = threadIdx.x; q < nloc; q += SMALL_THR) {
            const double xv = double(sX[q]);
            sZ[q] = c == 0.0 ? T(xv) : T(fma(-c, double(sG[q]), xv));
        }
        cl.sync();
    };
    auto adopt = [&](bool with_x) {  // (x, g) <- (z, g2): owned pixels only, by the thread that owns them
#pragma unroll
        for (int kk = 0; kk < PPT; ++kk) {
            const int q = threadIdx.x + kk * SMALL_THR;
            if (q >= nloc) break;
            if (with_x) sX[q] = sZ[q];
            sG[q] = g2[kk];
        }
        moved = moved || with_x;
    };

    // pass 0: gradient of x^{k,0} with f and ||g||^2
    double fx, s;
    {
        double v[2];
        small_terms<T, true, PPT>(sX, prev_last(sX), next_first(sX), r0, r1, ny, nx, v[0], v[1], g2, pij);
        small_reduce<2>(cl, sh, parity, v);
        adopt(false);
        fx = v[0];
        s = sqrt(v[1]);
        if (!isfinite(fx)) fault |= 2;
    }
    const double f_start = fx;
    const T* zp = prev_last(sZ);
    const T* zn = next_first(sZ);
    if (A.step_rule == SUP_RULE_ADAPTIVE) {
        // Eq. 11 (A-30): x <- x - ((f - f_ref)/||g||^2) g while f > f_ref and g != 0; no trial loop
        for (int nred = 0; nred < A.N; ++nred) {
            const bool take = fx > f_ref && s > 0.0;
            log_trial(f_ref, fx, take);
            if (!take) continue;
            ++trials;
            form_z(((fx - f_ref) / s) / s);
            if (nred == A.N - 1) {  // f and g of the final point are not needed
                for (int q = threadIdx.x; q < nloc; q += SMALL_THR) sX[q] = sZ[q];
                moved = true;
                break;
            }
            double v[2];
            small_terms<T, true, PPT>(sZ, zp, zn, r0, r1, ny, nx, v[0], v[1], g2, pij);
            small_reduce<2>(cl, sh, parity, v);
            adopt(true);
            fx = v[0];
            s = sqrt(v[1]);
            if (!isfinite(fx)) fault |= 2;
        }
    } else {
        for (int nred = 0; nred < A.N; ++nred) {
            const bool last = nred == A.N - 1;
            bool accepted = false;
            long long jloc = 0;
            int trial = 0;
            {   // the first candidate alone; when the step is not the last, with its gradient (accepted, the next step starts at once)
                const double c = step_coef(s, jloc);
                form_z(c);
                double v[2];
                const bool with_grad = !last;
                if (with_grad) {
                    small_terms<T, true, PPT>(sZ, zp, zn, r0, r1, ny, nx, v[0], v[1], g2, pij);
                    small_reduce<2>(cl, sh, parity, v);
                } else {
                    small_terms<T, false, PPT>(sZ, zp, zn, r0, r1, ny, nx, v[0], v[1], g2, pij);
                    small_reduce<1>(cl, sh, parity, v);
                }
                const bool acc = v[0] <= fx;  // NaN compares false -> rejected (A-11)
                ++ell;
                apow *= A.a;
                ++jloc;
                ++trials;
                ++trial;
                log_trial(v[0], fx, acc);
                if (acc) {
                    accepted = true;
                    if (last) {  // nobody needs the gradient at the final point
                        if (c != 0.0) {
                            for (int q = threadIdx.x; q < nloc; q += SMALL_THR) sX[q] = sZ[q];
                            moved = true;
                        }
                        fx = v[0];
                    } else {
                        fx = v[0];
                        s = sqrt(v[1]);
                        adopt(c != 0.0);
                    }
                }
            }
            // after a rejection: SMALL_NB candidates per pass, values only, decided strictly in order (later ones are discarded uncounted)
            while (!accepted && trial < SUP_J_MAX) {
                double coef[SMALL_NB], F[SMALL_NB];
                {
                    double ap = apow;
                    if (A.policy != SUP_STEP_PER_TRIAL) {
                        ap = 1.0;
                        for (long long q = 0; q < k + jloc; ++q) ap *= A.a;
                    }
#pragma unroll
                    for (int b = 0; b < SMALL_NB; ++b) {
                        coef[b] = s > 0.0 ? (A.beta0 * ap) / s : 0.0;
                        ap *= A.a;
                    }
                }
                small_terms_batch<T>(sX, sG, next_first(sX), next_first(sG), r0, r1, ny, nx, coef, F);
                small_reduce<SMALL_NB>(cl, sh, parity, F);
                double cacc = 0.0, facc = 0.0;
                for (int b = 0; b < SMALL_NB && !accepted && trial < SUP_J_MAX; ++b) {
                    const bool acc = F[b] <= fx;
                    ++ell;
                    apow *= A.a;
                    ++jloc;
                    ++trials;
                    ++trial;
                    log_trial(F[b], fx, acc);
                    if (acc) {
                        accepted = true;
                        cacc = coef[b];
                        facc = F[b];
                    }
                }
                if (!accepted) continue;
                form_z(cacc);
                if (last) {
                    if (cacc != 0.0) {
                        for (int q = threadIdx.x; q < nloc; q += SMALL_THR) sX[q] = sZ[q];
                        moved = true;
                    }
                    fx = facc;
                } else {  // the gradient at the accepted z (f(z) again: the same bits)
                    double v[2];
                    small_terms<T, true, PPT>(sZ, zp, zn, r0, r1, ny, nx, v[0], v[1], g2, pij);
                    small_reduce<2>(cl, sh, parity, v);
                    fx = v[0];
                    s = sqrt(v[1]);
                    adopt(cacc != 0.0);
                }
            }
            if (!accepted) warn |= 1;  // A-12: step skipped
        }
    }
    // the final iterate back to the caller's x and to the gather mirror of the product kernels
    if (moved || A.xg) {
        for (int q = threadIdx.x; q < nloc; q += SMALL_THR) {
            const T v = sX[q];
            if (moved) A.x[g0 + q] = v;
            if (A.xg) A.xg[sup_gmap(A.xmap, int(g0 + q))] = v;
        }
    }
    if (me == 0 && threadIdx.x == 0) {
        st->ell = ell;
        st->apow = apow;
        st->n_dec = ndec;
        st->n_trials += trials;
        st->sweep_trials += trials;
        st->f = fx;
        if (A.step_rule == SUP_RULE_ADAPTIVE && f_start <= f_ref) st->f_ref = A.shrink * f_start;  // A-30
        if (warn) atomicOr(&st->warn, warn);
        if (fault) atomicOr(&st->fault, fault);
    }
    cl.sync();  // no CTA leaves while another may still read its shared memory
}

// cluster size for an ny x nx image: 8, or 16 for more than 8 192 pixels when the device takes the non-portable size; 0: not eligible
static int small_cluster_size(const sup_ctx* h, int64_t ny, int64_t nx) {
    if (ny < SMALL_C || nx < 1 || ny * nx > int64_t(SMALL_C) * SMALL_LOCAL_MAX) return 0;
    int c = SMALL_C;
    if (ny * nx > 8192 && ny >= SMALL_CMAX && h->cluster16 > 0) c = SMALL_CMAX;
    const int64_t rows_max = (ny + c - 1) / c;
    return rows_max * nx <= SMALL_LOCAL_MAX ? c : 0;
}

bool sup_perturb_small_eligible(const sup_ctx* h, const PerturbParams& pp) {
    if (pp.objective != SUP_OBJ_TV2D || h->perturb_mode != 0) return false;
    return small_cluster_size(h, pp.ny, pp.nx) > 0;
}

template <typename T>
static sup_status launch_small_t(sup_ctx* h, const PArgs<T>& A, const PerturbParams& pp) {
    // (cluster16 must be known before the cluster size: ask with the general build's function once)
    const void* fn8 = reinterpret_cast<const void*>(&k_perturb_tv2d_small<T, SMALL_PPT>);
    const void* fn2 = reinterpret_cast<const void*>(&k_perturb_tv2d_small<T, 2>);
    const void* fn = fn8;
    if (!h->smem_opted_in.count(fn)) {
        SUP_CUDA(h, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, int(size_t(3) * SMALL_LOCAL_MAX * sizeof(T))));
        // does this device take clusters of 16 for this kernel?  (asked once per handle; -1 = no)
        h->cluster16 = -1;
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
            cudaLaunchConfig_t q = {};
            q.gridDim = dim3(SMALL_CMAX);
            q.blockDim = dim3(SMALL_THR);
            q.dynamicSmemBytes = size_t(3) * SMALL_LOCAL_MAX * sizeof(T);
            cudaLaunchAttribute qa[1];
            qa[0].id = cudaLaunchAttributeClusterDimension;
            qa[0].val.clusterDim.x = SMALL_CMAX;
            qa[0].val.clusterDim.y = 1;
            qa[0].val.clusterDim.z = 1;
            q.attrs = qa;
            q.numAttrs = 1;
            int nclusters = 0;
            if (cudaOccupancyMaxActiveClusters(&nclusters, fn, &q) == cudaSuccess && nclusters >= 1) h->cluster16 = 1;
        }
        cudaFuncSetAttribute(fn2, cudaFuncAttributeMaxDynamicSharedMemorySize, int(size_t(3) * SMALL_LOCAL_MAX * sizeof(T)));
        if (h->cluster16 > 0) cudaFuncSetAttribute(fn2, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        cudaGetLastError();
        h->smem_opted_in.insert(fn);
    }
    const int C = small_cluster_size(h, pp.ny, pp.nx);
    if (C < 1) return sup_fail(h, SUP_ERR_STATE, "sup_launch_perturb_small: image not eligible");
    const int rows_max = int((pp.ny + C - 1) / C);
    const size_t smem = size_t(3) * rows_max * pp.nx * sizeof(T);
    if (int64_t(rows_max) * pp.nx <= 2 * SMALL_THR) fn = fn2;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C);
    cfg.blockDim = dim3(SMALL_THR);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    PArgs<T> Ac = A;
    int rm = rows_max;
    void* args[] = {&Ac, &rm};
    SUP_CUDA(h, cudaLaunchKernelExC(&cfg, fn, args));
    h->launches++;
    return SUP_OK;
}

sup_status sup_launch_perturb_small(sup_ctx* h, void* x, const PerturbParams& pp) {
    if (h->dt == SUP_F32) return launch_small_t<float>(h, sup_make_perturb_args<float>(h, x, pp), pp);
    return launch_small_t<double>(h, sup_make_perturb_args<double>(h, x, pp), pp);
}
