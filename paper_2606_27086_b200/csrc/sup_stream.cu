// sup_stream.cu -- S1+S2 and S3 of the hot path as persistent kernels whose val/col stream is
// staged through shared memory by the bulk-copy engine.
//
//   S1+S2  r_i = <a_i, x>, c_i = hyperslab violation (Eq. 2 on each face, L38-42; Eq. 20),
//          y_i = d_i c_i, d_i = w_i/||a_i||^2 (L608)
//   S3     u_j = sum_i a_ij y_i over row j of the explicit A^T,  x_j <- clip(x_j - lambda u_j) (Eq. 3; box L427)
//
// Why: ncu on the group-per-row kernels (profiles/r01a_spmv_baseline.md) shows DRAM traffic equal to the algorithmic
// bytes but only 57-60 % of the measured copy bandwidth with nothing saturated; the L1 fills (stream + gather
// misses, 3.35 GB per launch) all go through the LSU miss path.  Two earlier attempts are recorded in
// profiles/r01b_ring_negative.md.  This version takes the stream off the LSU path:
//   * one persistent CTA per SM owns a CONTIGUOUS row range balanced by cost (nonzeros + a constant per row;
//     partition table built at setup), hence a contiguous range of the matrix stream;
//   * fp32 handles stream PACKED (value bits, column) pairs -- one cp.async.bulk per 8 KB tile, one 64-bit shared
//     load per element (the copy engine costs ~72 cycles per copy, profiles/r01e_packed.md); fp64 handles stream
//     val[] and col[] as two copies per tile;
//   * a producer thread pulls the range through a ring of tiles in shared memory (20 stages for the fp32 forward
//     product, 16 otherwise), L2 evict-first, completing on per-stage mbarriers; the stream never occupies L1,
//     which is left to the x / y gathers, and it announces each armed stage in issued[];
//   * the consumer warps (12 by default) take the rows in order (G lanes per row; G = 64: a warp pair per row;
//     G = 0: the whole CTA per row, for rows of thousands of entries), wait on the barriers of the tiles their rows
//     span, read the ring (consecutive lanes -> consecutive words), gather x / y through L1 (ld.global.nc, 16 in
//     flight per lane), reduce with shuffles and run the fused epilogue.  Each consumer warp publishes how many
//     tiles lie wholly before its rows; the producer refills a stage when every warp has passed it.
// The forward product gathers from xg, the bank-swizzled mirror of x (sup_swz), which the back-projection keeps
// in step.  The summation order of a row depends only on G, not on the grid: results are deterministic.
#include <math.h>
#include <stdlib.h>

#include "sup_internal.cuh"

#ifndef RG_TILE
#define RG_TILE 1024                        // elements per stage
#endif
// Shape of the persistent CTA: consumer warps NCW and ring stages STG (fp32 tiles are 8 KB of packed pairs, fp64 tiles
// 12 KB of separate val / col).  More warps in flight hide more gather latency, but the rows they hold at once take ring
// stages away from the prefetch, and the ring takes shared memory away from the L1 the gathers live in.  Two shapes per
// direction (profiles/r02e_sweep.md, config 3):
//   DEEP  -- the gathered vector has a tiled layout (sup_set_layout: its working set in L1 is ~2.6x smaller): 24 stages
//            (the most that keeps the 196 KB shared-memory carve-out; 25 fall off a cliff), 14 / 18 warps forward / backward
//   BASE  -- no layout known: round 1's shape, 12 warps, 20 stages forward / 16 backward (a deeper ring starves the L1)
// fp64 handles: BASE warps with 16 stages (192 KB).
#define RG_STAGES_MIN 16                    // what the planner may count on in every instantiation
template <typename T, int MODE, bool DEEP>
struct RgShape {
    static constexpr int NCW = !DEEP || sizeof(T) != 4 ? 12 : (MODE == 0 ? 14 : 18);
    static constexpr int STG = sizeof(T) != 4 ? 16 : (DEEP ? 24 : (MODE == 0 ? 20 : 16));
};
#define RG_NCARRY 256
#ifndef RG_SEG_MIN_AVG
#define RG_SEG_MIN_AVG 1e300                // mean row length from which the planner would pick the segment mode (G = 1): never --
                                            // it is correct but 1.7-3.7x slower than the row modes (profiles/r02j_segments.md); sup_set_row_mode(h, 1, 1) selects it
#endif
// G == 128 (chunks of long rows): pool of chunk partial sums and row counters; see the consumer branch for the bounds
#define RG_CHUNK_POOL 256
#define RG_CHUNK_ROWS 64
#define RG_CHUNK_KMAX 128
static_assert(sizeof(float) * RG_CHUNK_POOL + 4 * RG_CHUNK_ROWS <= 8 * RG_NCARRY, "the chunk pool must fit the carry slots' space");
#define RG_CWARPS 24                        // upper bound on the consumer warps (sizes of the shared arrays)
#ifndef RG_NPROD
#define RG_NPROD 2                          // producer warps: ONE thread issues at most one bulk copy per ~270 ns whatever its size
#endif                                      // (profiles/r02b_producer.md), i.e. 4.5 TB/s of 8 KB tiles chip-wide; two reach the HBM rate
#ifndef RG_UNROLL
#define RG_UNROLL 16                        // independent gathers in flight per lane (a multiple of 4)
#endif
#ifndef RG_SPIN_SLEEP_C
#define RG_SPIN_SLEEP_C 0                  // ns a consumer sleeps between polls of issued[] (0: busy poll)
#endif
#ifndef RG_SPIN_SLEEP_P
#define RG_SPIN_SLEEP_P 0                  // ns a producer sleeps between polls of the consumers' progress
#endif
#define RG_TIMEOUT 8000000000LL             // ~4 s of SM clocks: a protocol bug must fault, not hang the GPU

// ---- PTX wrappers (mbarrier + bulk copy) --------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok = 0;
    long long t0 = 0;
    for (;;) {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (t0 == 0) t0 = clock64();
        else if (clock64() - t0 > RG_TIMEOUT) __trap();
    }
}
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}

#ifdef SUP_PROFILE
__device__ unsigned long long g_prof[8];  // G == 1 also: 6 carry wait, 7 accumulate phase  // 0 consumer data-wait, 1 consumer dot, 2 consumer total, 3 producer free-wait, 4 producer total, 5 kernel
#define PROF_T(v) const long long v = clock64()
#define PROF_DECL long long prof_acc[6] = {0, 0, 0, 0, 0, 0}
#define PROF_ADD(i, d) prof_acc[i] += (long long)(d)
#define PROF_FLUSH(i) do { if (lane == 0) atomicAdd(&g_prof[i], (unsigned long long)prof_acc[i]); } while (0)
extern "C" void sup_prof_read(unsigned long long* out, int reset) {
    cudaMemcpyFromSymbol(out, g_prof, sizeof(g_prof));
    if (reset) { unsigned long long z[8] = {0}; cudaMemcpyToSymbol(g_prof, z, sizeof(z)); }
}
#else
#define PROF_T(v)
#define PROF_DECL
#define PROF_ADD(i, d)
#define PROF_FLUSH(i)
#endif

template <typename T>
__device__ __forceinline__ T hyperslab_violation(T r, T lb, T ub) {  // Eq. 2 on each face of lb <= r <= ub
    return r > ub ? r - ub : (r < lb ? r - lb : T(0));
}

// Ring storage.  fp64: separate val / col arrays (two bulk copies per tile).  fp32: PACKED (value bits, column) pairs,
// one 8-byte word per nonzero, so a tile is ONE bulk copy and a consumer needs one 64-bit shared load per element.
// (Measured on config 3: the bulk-copy engine costs ~72 cycles per copy on top of ~0.043 cycles per byte -- the same
// bytes as twice as many copies ran 23-25 % slower, profiles/r01e_packed.md -- so fewer, larger copies matter.)
template <typename T, int STG>
struct RgData {
    T val[STG * RG_TILE];
    int32_t col[STG * RG_TILE];
};
template <int STG>
struct RgData<float, STG> {
    uint2 pair[STG * RG_TILE];
};
template <int STG>
__device__ __forceinline__ void ring_get(const RgData<double, STG>& d, int i, int& c, double& v) {
    c = d.col[i];
    v = d.val[i];
}
template <int STG>
__device__ __forceinline__ void ring_get(const RgData<float, STG>& d, int i, int& c, float& v) {
    const uint2 q = d.pair[i];
    v = __uint_as_float(q.x);
    c = int(q.y);
}

template <typename T>
struct CarrySlot;
template <>
struct CarrySlot<float> {
    typedef unsigned long long type;  // value bits | flag << 32
    static __device__ __forceinline__ void put(volatile type* p, float v, int flag) { *p = (type(unsigned(flag)) << 32) | type(__float_as_uint(v)); }
    static __device__ __forceinline__ bool get(volatile type* p, int flag, float& v) {
        const type w = *p;
        v = __uint_as_float(unsigned(w));
        return int(w >> 32) == flag;
    }
};
template <>
struct CarrySlot<double> {
    typedef ulonglong2 type;  // .x value bits, .y flag: one 16-byte shared access
    static __device__ __forceinline__ void put(volatile type* p, double v, int flag) {
        asm volatile("st.volatile.shared.v2.b64 [%0], {%1, %2};" ::"r"(smem_u32(const_cast<type*>(p))), "l"(__double_as_longlong(v)), "l"((long long)flag) : "memory");
    }
    static __device__ __forceinline__ bool get(volatile type* p, int flag, double& v) {
        long long a, b;
        asm volatile("ld.volatile.shared.v2.b64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "r"(smem_u32(const_cast<type*>(p))) : "memory");
        v = __longlong_as_double(a);
        return int(b) == flag;
    }
};

template <typename T, int STG>
struct RgSmem {
    RgData<T, STG> d;
    unsigned long long full[STG];
    T ctabuf[2][RG_CWARPS];       // G == 0: the consumer warps' partial sums of one long row (double-buffered by row parity)
    T pairbuf[RG_CWARPS / 2][2];  // G == 64: partial row sums handed from the odd to the even warp of a pair
    int progress[RG_CWARPS];  // per consumer warp: tiles [0, progress) are no longer needed by it
    int issued[STG];          // per stage: 1 + the tile its barrier is currently armed for (0: none yet)
    double red[RG_CWARPS];    // per consumer warp: its share of the kernel's reduction
    // G == 1: slot s mod RG_NCARRY = (partial sum of the row left open at the end of segment s, 1 + s), written and read as ONE
    // vector access so that no fence is needed between value and flag
    // G == 128: partial sums of the chunks of multi-chunk rows (a pool indexed by the running chunk number) and one arrival
    // counter per such row; shares its space with the carry slots (never both in one kernel)
    union {
        typename CarrySlot<T>::type carry[RG_NCARRY];
        struct {
            T part[RG_CHUNK_POOL];
            int cnt[RG_CHUNK_ROWS];
        } ck;
    };
};

// Dot product of the ring elements k, k+G, k+2G, ... < e (offsets relative to the stream base) with gathered vec
// entries, RG_UNROLL independent gathers in flight per lane.  Element u of a lane always goes to accumulator u mod 4, so the
// result does not depend on where the row sits in the ring.  WRAP: the row crosses the end of the ring.
template <typename T, int G, bool WRAP, int STG>
__device__ __forceinline__ void ring_row_dot(const RgData<T, STG>& ring, const T* __restrict__ vec, int k, int e,
                                             int trips, volatile int* prog, int rel_tiles, bool lane0,
                                             T& a0, T& a1, T& a2, T& a3) {
    int n = e - k;  // this lane's elements are k, k+G, ... while offset < n
    constexpr int RG_ELEMS = STG * RG_TILE;
    int p = k % RG_ELEMS;
    // `trips` is warp-uniform (the longest row of the warp decides); lanes whose row is exhausted run predicated off
    for (int trip = 0; trip < trips; ++trip, n -= RG_UNROLL * G, p += RG_UNROLL * G) {
        if (WRAP && p >= RG_ELEMS) p -= RG_ELEMS;
        int c[RG_UNROLL];
        T v[RG_UNROLL], g[RG_UNROLL];
        const bool full = n > (RG_UNROLL - 1) * G;
        if (full) {
#pragma unroll
            for (int u = 0; u < RG_UNROLL; ++u) {
                int i = p + u * G;
                if (WRAP && i >= RG_ELEMS) i -= RG_ELEMS;
                ring_get(ring, i, c[u], v[u]);
            }
        } else {  // last, partial group (or nothing left): predicated
#pragma unroll
            for (int u = 0; u < RG_UNROLL; ++u) {
                const bool in = u * G < n;
                int i = in ? p + u * G : 0;
                if (WRAP && i >= RG_ELEMS) i -= RG_ELEMS;
                ring_get(ring, i, c[u], v[u]);  // (index 0 when out of range)
                c[u] = in ? c[u] : 0;
                v[u] = in ? v[u] : T(0);
            }
        }
        if (trip == trips - 1) {
            // Early release: the warp has read everything it needs from the ring for these rows, so the tiles wholly
            // before the end of its rows can be refilled while the gathers below are still in flight.
            __syncwarp();
            if (lane0) *prog = rel_tiles;
        }
        if (full) {
#pragma unroll
            for (int u = 0; u < RG_UNROLL; ++u) g[u] = __ldg(vec + c[u]);
        } else {
#pragma unroll
            for (int u = 0; u < RG_UNROLL; ++u) g[u] = (u * G < n) ? __ldg(vec + c[u]) : T(0);
        }
#pragma unroll
        for (int u = 0; u < RG_UNROLL; u += 4) {
            a0 += v[u] * g[u];
            a1 += v[u + 1] * g[u + 1];
            a2 += v[u + 2] * g[u + 2];
            a3 += v[u + 3] * g[u + 3];
        }
    }
}

// Fused epilogue of one finished row r, run by ONE lane; racc collects the row's term of the kernel's fp64 reduction.
//   MODE 0  y_r = q3 * c,  c = hyperslab violation of the row value against [q1, q2]  (Eq. 2 per face; q3 = d_r or w_r);
//           reduction: sum c * y  (= sum w_i c_i^2 / ||a_i||^2 when q3 = d: Eq. 12 with p = 2, twice Eq. 5)
//   MODE 1  x_r <- clip(x_r - lambda * q4 * u_r, q1, q2)  (Eq. 3, box L427; q4 = 1, or DROP's 1/nnz(A_:,r)); mirror in out2
//   MODE 2  out_r = lambda * (row value)  (a plain product with a scale);  reduction: sum q3 * out_r^2  (q3 = 1 or a weight)
template <typename T, int MODE>
__device__ __forceinline__ void row_epilogue(int64_t r, T acc, T q1, T q2, T q3, T q4, T* out, T* out2, T lambda, const GMap& omap,
                                             double& racc) {
    if (MODE == 0) {
        const T c = hyperslab_violation(acc, q1, q2);
        const T y = q3 * c;
        out[sup_gmap(omap, int(r))] = y;  // (in y's gather layout)
        racc += double(c) * double(y);
    } else if (MODE == 1) {
        T t = q3 - lambda * (q4 * acc);  // Eq. 3
        t = t < q1 ? q1 : t;             // box, un-relaxed (A-2)
        t = t > q2 ? q2 : t;
        out[r] = t;
        if (out2) out2[sup_gmap(omap, int(r))] = t;  // keep the gather mirror of x in step
    } else {
        const T v = lambda * acc;
        out[sup_gmap(omap, int(r))] = v;
        racc += double(q3) * (double(v) * double(v));
    }
}
// loads the compiler may not sink towards their use (the segment mode issues a row's operands long before the row's
// sum is complete, and the use sits on the carry chain between segments, where an L2 round trip would serialise the warps)
__device__ __forceinline__ float ld_pinned(const float* p) {
    float v;
    asm volatile("ld.global.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ double ld_pinned(const double* p) {
    double v;
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}
template <typename T, int MODE>
__device__ __forceinline__ void row_operands_pinned(int64_t r, const T* p1, const T* p2, const T* p3, const T* out, T& q1, T& q2, T& q3, T& q4) {
    q4 = T(1);
    if (MODE == 0) {
        q1 = ld_pinned(p1 + r);
        q2 = ld_pinned(p2 + r);
        q3 = ld_pinned(p3 + r);
    } else if (MODE == 1) {
        q1 = ld_pinned(p1 + r);
        q2 = ld_pinned(p2 + r);
        q3 = ld_pinned(out + r);
        if (p3) q4 = ld_pinned(p3 + r);
    } else {
        q1 = q2 = T(0);
        q3 = p3 ? ld_pinned(p3 + r) : T(1);
    }
}

template <typename T, int MODE>
__device__ __forceinline__ void row_operands(int64_t r, const T* p1, const T* p2, const T* p3, const T* out, T& q1, T& q2, T& q3, T& q4) {
    q4 = T(1);
    if (MODE == 0) {
        q1 = p1[r];
        q2 = p2[r];
        q3 = p3[r];
    } else if (MODE == 1) {
        q1 = p1[r];
        q2 = p2[r];
        q3 = out[r];
        if (p3) q4 = p3[r];
    } else {
        q1 = q2 = T(0);
        q3 = p3 ? p3[r] : T(1);
    }
}

// MODE 0: forward (vec = xg, columns swizzled (pk / colg), p1 = lb, p2 = ub, p3 = d, out = y);
// MODE 1: backward (vec = y, p1 = lo, p2 = hi, out = x in place, out2 = xg mirror or NULL)
// Programmatic dependent launch (sm_90+): k_staged launches are given the programmatic-serialization attribute.  Every CTA allows its dependents to launch as soon as it has started; a dependent CTA becomes
// resident on an SM the moment the earlier kernel's CTA there exits (one CTA per SM: the ring owns the shared memory), its PRODUCERS
// start streaming the matrix (static data) into the ring at once, its CONSUMERS first wait for the earlier grid to complete and flush
// (they read x / y, which it writes).  The launch latency, the ring fill and the earlier kernel's tail (CTAs finish unevenly)
// overlap; block-iterative sweeps have 32 such boundaries per sweep.  Without the attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename T, int MODE, int G, int NCW, int STG>
__global__ void __launch_bounds__(32 * (NCW + RG_NPROD), 1)
    k_staged(const int64_t* __restrict__ part, const int64_t* __restrict__ rowptr, const int32_t* __restrict__ col,
             const T* __restrict__ val, const uint2* __restrict__ pk, const T* __restrict__ vec, const T* __restrict__ p1,
             const T* __restrict__ p2, const T* __restrict__ p3, T* out, T* out2, T lambda, int64_t nnz_total, const GMap omap, double* __restrict__ red_out,
             const int* __restrict__ stop) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int RG_ELEMS = STG * RG_TILE;
    RgSmem<T, STG>& S = *reinterpret_cast<RgSmem<T, STG>*>(smem_raw);
    if (stop && *stop) return;  // the stopping rule fired earlier in this run (A-25): the sweep is skipped (no PDL with a stop flag)
    pdl_launch_dependents();
    const int64_t rs = part[blockIdx.x], re = part[blockIdx.x + 1];
    if (rs >= re) {
        pdl_wait();
        if (red_out && threadIdx.x == 0) red_out[blockIdx.x] = 0.0;
        return;
    }
    const int64_t es = rowptr[rs], ee = rowptr[re];
    const int64_t base = es & ~int64_t(3);  // 16-byte aligned start of the stream (4 elements)
    // an all-empty range streams nothing (no copy may be left in flight when the CTA exits)
    const int ntiles = ee > es ? int((ee - base + RG_TILE - 1) / RG_TILE) : 0;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STG; ++s) mbar_init(smem_u32(&S.full[s]), 1);
        for (int w = 0; w < NCW; ++w) S.progress[w] = 0;
        for (int st = 0; st < STG; ++st) S.issued[st] = 0;
        if constexpr (G == 128) {
            for (int q = 0; q < RG_CHUNK_ROWS; ++q) S.ck.cnt[q] = 0;
        } else {
            for (int q = 0; q < RG_NCARRY; ++q) CarrySlot<T>::put(&S.carry[q], T(0), 0);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    volatile int* progress = S.progress;
    volatile int* issued = S.issued;

    if (warp >= NCW) {
        // ---- producers: lane 0 of each producer warp feeds the ring, warp p the tiles t = p (mod RG_NPROD).  (More LANES
        // of one warp brought nothing in round 1 -- they serialise; separate warps issue in parallel.) ---------------------
        if (lane == 0) {
            const uint64_t pol = l2_evict_first_policy();
            const int64_t bulk_limit = nnz_total & ~int64_t(3);  // bulk copies never read past the arrays' last whole 16 B
            int freed = 0;                                        // min over the consumer warps' progress
            PROF_DECL;
            PROF_T(pt0);
            for (int t = warp - NCW; t < ntiles; t += RG_NPROD) {
                const int s = t % STG;
                if (t >= STG && freed <= t - STG) {
                    PROF_T(pw0);
                    const long long t0 = clock64();
                    for (;;) {
                        int mn = progress[0];
#pragma unroll
                        for (int w = 1; w < NCW; ++w) {
                            const int p = progress[w];
                            mn = p < mn ? p : mn;
                        }
                        freed = mn;
                        if (freed > t - STG) break;
                        if (RG_SPIN_SLEEP_P) __nanosleep(RG_SPIN_SLEEP_P);
                        if (clock64() - t0 > RG_TIMEOUT) __trap();
                    }
                    // the consumers' reads of the stage (generic proxy) precede the bulk write (async proxy)
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    PROF_ADD(3, clock64() - pw0);
                }
                const int64_t g0 = base + int64_t(t) * RG_TILE;
                const int64_t g1 = (g0 + RG_TILE < ee) ? g0 + RG_TILE : ee;  // elements needed: [g0, g1)
                int64_t gb = (g1 + 3) & ~int64_t(3);                          // bulk part: [g0, gb)
                if (gb > nnz_total) gb = bulk_limit > g0 ? bulk_limit : g0;
                constexpr bool PACKED = sizeof(T) == 4;
                for (int64_t g = gb; g < g1; ++g) {  // at most 3 ragged elements at the very end of the arrays
                    if constexpr (PACKED) {
                        S.d.pair[s * RG_TILE + int(g - g0)] = pk[g];
                    } else {
                        S.d.val[s * RG_TILE + int(g - g0)] = val[g];
                        S.d.col[s * RG_TILE + int(g - g0)] = col[g];
                    }
                }
                const uint32_t ne = uint32_t(gb - g0);
                const uint32_t bar = smem_u32(&S.full[s]);
                if (ne == 0) {
                    mbar_arrive(bar);
                } else if constexpr (PACKED) {
                    mbar_arrive_expect_tx(bar, ne * 8u);
                    bulk_g2s(smem_u32(&S.d.pair[s * RG_TILE]), pk + g0, ne * 8u, bar, pol);
                } else {
                    mbar_arrive_expect_tx(bar, ne * uint32_t(sizeof(T) + 4));
                    bulk_g2s(smem_u32(&S.d.val[s * RG_TILE]), val + g0, ne * uint32_t(sizeof(T)), bar, pol);
                    bulk_g2s(smem_u32(&S.d.col[s * RG_TILE]), col + g0, ne * 4u, bar, pol);
                }
                issued[s] = t + 1;  // the stage's barrier is armed for tile t: consumers may now wait on its phase
            }
            PROF_ADD(4, clock64() - pt0);
            PROF_FLUSH(3);
            PROF_FLUSH(4);
            // Do not leave while a copy may still be in flight into this CTA's shared memory (the consumers wait on every
            // tile their rows touch, but a tile holding only alignment padding or the tail of an empty row has no reader).
            // (each producer waits for the tiles it armed itself, so the phase parity is unambiguous)
            for (int t = ntiles > STG ? ntiles - STG : 0; t < ntiles; ++t)
                if (t % RG_NPROD == warp - NCW) mbar_wait(smem_u32(&S.full[t % STG]), (t / STG) & 1);
        }
        return;
    }
    double racc = 0.0;  // this lane's share of the kernel's reduction (row_epilogue)
    pdl_wait();         // the vectors this kernel gathers and updates are complete and visible from here on
    // ---- consumers, G == 0: LONG rows -- the whole CTA works on one row at a time ----------------------------------------
    // (rows of thousands of nonzeros, e.g. config 4's A^T: one row per warp would put NCW x row bytes in flight, far more
    // than the ring holds).  The row is cut into pieces of 32 NCW x RG_UNROLL elements; every lane takes RG_UNROLL elements
    // of a piece, tiles are released piece by piece, so the row length is unbounded; the warps' partial sums meet in shared
    // memory and warp 0 adds them in a fixed order.
    if constexpr (G == 0) {
        constexpr int GT = 32 * NCW;
        constexpr int CH = GT * RG_UNROLL;
        const int gl = warp * 32 + lane;
        int seen = 0, released = 0, iter = 0;
        int s = int(rowptr[rs] - base), e = int(rowptr[rs + 1] - base);
        for (int64_t r = rs; r < re; ++r, ++iter) {
            int s_next = 0, e_next = 0;
            if (r + 1 < re) {
                s_next = e;
                e_next = int(rowptr[r + 2] - base);
            }
            T q1 = T(0), q2 = T(0), q3 = T(0), q4 = T(1);
            if (gl == 0) row_operands<T, MODE>(r, p1, p2, p3, out, q1, q2, q3, q4);
            T a0 = T(0), a1 = T(0), a2 = T(0), a3 = T(0);
            for (int ps = s; ps < e; ps += CH) {
                const int pe = e < ps + CH ? e : ps + CH;
                int t_start = ps / RG_TILE;
                t_start = t_start < ntiles ? t_start : ntiles;
                if (released < t_start) {
                    released = t_start;
                    if (lane == 0) progress[warp] = t_start;
                }
                const int t_hi = (pe - 1) / RG_TILE;
                for (int t = seen > t_start ? seen : t_start; t <= t_hi; ++t) {
                    const int st = t % STG;
                    if (issued[st] != t + 1) {
                        const long long t0 = clock64();
                        while (issued[st] != t + 1) {
                            if (RG_SPIN_SLEEP_C) __nanosleep(RG_SPIN_SLEEP_C);
                            if (clock64() - t0 > RG_TIMEOUT) __trap();
                        }
                    }
                    mbar_wait(smem_u32(&S.full[st]), (t / STG) & 1);
                }
                seen = seen > t_hi + 1 ? seen : t_hi + 1;
                asm volatile("" ::: "memory");
                int rel = pe / RG_TILE;
                rel = rel < ntiles ? rel : ntiles;
                rel = rel > released ? rel : released;
                const bool wraps = (ps % RG_ELEMS) + (pe - ps) > RG_ELEMS;
                if (!wraps) ring_row_dot<T, GT, false, STG>(S.d, vec, ps + gl, pe, 1, progress + warp, rel, lane == 0, a0, a1, a2, a3);
                else ring_row_dot<T, GT, true, STG>(S.d, vec, ps + gl, pe, 1, progress + warp, rel, lane == 0, a0, a1, a2, a3);
                released = rel;
            }
            T acc = (a0 + a1) + (a2 + a3);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) S.ctabuf[iter & 1][warp] = acc;
            asm volatile("bar.sync 1, %0;" ::"n"(GT) : "memory");
            if (gl == 0) {
                T tot = T(0);
#pragma unroll
                for (int w = 0; w < NCW; ++w) tot += S.ctabuf[iter & 1][w];
                row_epilogue<T, MODE>(r, tot, q1, q2, q3, q4, out, out2, lambda, omap, racc);
            }
            s = s_next;
            e = e_next;
        }
        __syncwarp();
        if (lane == 0) progress[warp] = ntiles;
    } else if constexpr (G == 128) {
    // ---- consumers, G == 128: CHUNKS of long rows (rows of thousands of entries: config 4's A^T) -----------------------------------
    // A row of len elements is K = ceil(len / CHK) chunks of CHK = 32 x RG_UNROLL elements, aligned to the row's start; the chunks of
    // the CTA's rows, numbered in stream order, go to the warps round-robin (chunk u to warp u mod NCW).  Every trip but a row's last
    // is full, no warp waits for another, and the ring span of the warps in flight is NCW chunks whatever the row lengths.  A warp
    // leaves its chunk's sum in the pool (slot = running chunk number of the multi-chunk rows, mod RG_CHUNK_POOL) and counts itself
    // in on the row's counter; the warp that arrives last adds the K sums IN CHUNK ORDER and runs the epilogue, so the row value does
    // not depend on the timing.  Bounds: a multi-chunk row has more than CHK (K - 1) elements and the warps are at most one ring
    // (<= 24 576 elements) apart, so at most 48 multi-chunk rows and 96 + K pool slots are live at once: RG_CHUNK_ROWS = 64,
    // K <= RG_CHUNK_KMAX = 128 (the planner checks the longest row) with RG_CHUNK_POOL = 256.
        constexpr int CHK = 32 * RG_UNROLL;
        int seen = 0, released = 0;
        int u0 = 0;  // chunks before row r (all rows)
        int mc = 0;  // chunks before row r, multi-chunk rows only
        int mr = 0;  // multi-chunk rows before row r
        int64_t rp = rowptr[rs];
        for (int64_t r = rs; r < re; ++r) {
            const int s = int(rp - base);
            rp = rowptr[r + 1];
            const int e = int(rp - base);
            const int K = (e - s + CHK - 1) / CHK;
            if (K == 0) {  // empty row: its epilogue by one lane of one warp
                if (int((r - rs) % NCW) == warp && lane == 0) {
                    T q1, q2, q3, q4;
                    row_operands<T, MODE>(r, p1, p2, p3, out, q1, q2, q3, q4);
                    row_epilogue<T, MODE>(r, T(0), q1, q2, q3, q4, out, out2, lambda, omap, racc);
                }
                continue;
            }
            int c = (warp - u0 % NCW + NCW) % NCW;  // this warp's first chunk of the row
            for (; c < K; c += NCW) {
                const int ps = s + c * CHK;
                const int pe = e < ps + CHK ? e : ps + CHK;
                int t_start = ps / RG_TILE;
                t_start = t_start < ntiles ? t_start : ntiles;
                if (released < t_start) {
                    released = t_start;
                    if (lane == 0) progress[warp] = t_start;
                }
                const int t_hi = (pe - 1) / RG_TILE;
                for (int t = seen > t_start ? seen : t_start; t <= t_hi; ++t) {
                    const int st = t % STG;
                    if (issued[st] != t + 1) {
                        const long long t0 = clock64();
                        while (issued[st] != t + 1)
                            if (clock64() - t0 > RG_TIMEOUT) __trap();
                    }
                    mbar_wait(smem_u32(&S.full[st]), (t / STG) & 1);
                }
                seen = seen > t_hi + 1 ? seen : t_hi + 1;
                asm volatile("" ::: "memory");
                int rel = pe / RG_TILE;
                rel = rel < ntiles ? rel : ntiles;
                rel = rel > released ? rel : released;
                T a0 = T(0), a1 = T(0), a2 = T(0), a3 = T(0);
                const bool wraps = (ps % RG_ELEMS) + (pe - ps) > RG_ELEMS;
                if (!wraps) ring_row_dot<T, 32, false, STG>(S.d, vec, ps + lane, pe, 1, progress + warp, rel, lane == 0, a0, a1, a2, a3);
                else ring_row_dot<T, 32, true, STG>(S.d, vec, ps + lane, pe, 1, progress + warp, rel, lane == 0, a0, a1, a2, a3);
                released = rel;
                T acc = (a0 + a1) + (a2 + a3);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
                if (lane == 0) {
                    bool finish = K == 1;
                    T tot = acc;
                    if (K > 1) {
                        volatile T* pool = S.ck.part;
                        pool[(mc + c) % RG_CHUNK_POOL] = acc;
                        __threadfence_block();
                        const int arrived = atomicAdd(&S.ck.cnt[mr % RG_CHUNK_ROWS], 1);
                        if (arrived == K - 1) {  // the last chunk to arrive: add the K sums in chunk order
                            __threadfence_block();
                            tot = T(0);
                            for (int q = 0; q < K; ++q) tot += pool[(mc + q) % RG_CHUNK_POOL];
                            S.ck.cnt[mr % RG_CHUNK_ROWS] = 0;
                            finish = true;
                        }
                    }
                    if (finish) {
                        T q1, q2, q3, q4;
                        row_operands<T, MODE>(r, p1, p2, p3, out, q1, q2, q3, q4);
                        row_epilogue<T, MODE>(r, tot, q1, q2, q3, q4, out, out2, lambda, omap, racc);
                    }
                }
            }
            u0 += K;
            if (K > 1) {
                mc += K;
                ++mr;
            }
        }
        __syncwarp();
        if (lane == 0) progress[warp] = ntiles;
    } else if constexpr (G == 1) {
    // ---- consumers, G == 1: SEGMENTS of the stream instead of rows (rows of hundreds of entries and more) ---------------------
    // Warp w takes the segments w, w + NCW, ... of 32 x RG_UNROLL consecutive elements of the CTA's stream, whatever rows they belong
    // to: every trip is full (no predicated partial groups), there is no per-row prologue, and the ring span of the warps in flight
    // is NCW segments whatever the row lengths.  Lane l holds the elements S0 + 32 u + l; a group of 32 consecutive elements lies
    // inside one row unless a row END falls into it (a warp-uniform test per group); where one does, the lanes before it finish
    // that row: warp sum, plus the partial sum carried over from earlier segments, epilogue by the lane that prefetched the row's
    // operands.  The sum of what follows the last row end of a segment is handed to the next segment through shared memory
    // (carry[], in segment order: a fixed summation order).  Row ends are found in a window of 32 consecutive row pointers that
    // each warp keeps sliding forward (loaded one segment ahead).
        constexpr int SEG = 32 * RG_UNROLL;
        static_assert(RG_TILE % SEG == 0, "a segment must not straddle two ring stages' end");
        const unsigned FULLM = 0xffffffffu;
        const int E = int(ee - base), F = int(es - base);  // valid elements of the stream: [F, E)
        const int nseg = E > 0 ? (E + SEG - 1) / SEG : 1;  // (an all-empty range still has its rows to write)
        volatile typename CarrySlot<T>::type* carry = S.carry;
        auto load_window = [&](int64_t r) -> int {  // lane l: end of row r + l as a stream offset (rows beyond the range never end)
            const int64_t rr = r + lane;
            return rr < re ? int(rowptr[rr + 1] - base) : 0x7fffffff;
        };
        auto warp_sum = [&](T v) -> T {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULLM, v, o);
            return v;
        };
        int64_t wrow = rs;               // first row of the window; rows before it are finished
        int wend = load_window(wrow);
        int seen = 0, released = 0;
        // The first row that ends in a segment began in an earlier one: its sum needs the carry of the segment before.  Nothing else
        // does -- in particular not the segment's own carry-out when a row ends in it -- so that row is parked (head_*) and only
        // completed one segment of this warp later, when the carry has long been published: the warps never wait for each other
        // except through segments no row ends in (rows longer than a segment).
        bool head_pending = false;
        T head_sum = T(0);
        int head_lane = 0, head_seg = 0;
        int64_t head_row = 0;
        T hq1 = T(0), hq2 = T(0), hq3 = T(0), hq4 = T(1);
        PROF_DECL;
        PROF_T(ct0);
        for (int sg = warp; sg < nseg; sg += NCW) {
            PROF_T(it0);
            const int S0 = sg * SEG;
            const int S1 = S0 + SEG < E ? S0 + SEG : E;
            // rows that ended at or before S0 were finished by earlier segments (segment 0: leading empty rows are its own)
            int nskip = 0;
            if (sg > 0) {
                for (;;) {
                    nskip = __popc(__ballot_sync(FULLM, wend <= S0));
                    if (nskip < 32) break;
                    wrow += 32;
                    wend = load_window(wrow);
                }
            }
            int jb = nskip;  // window lane of the next row to finish
            int e_next = __shfl_sync(FULLM, wend, jb);
            // Row-end window for this warp's NEXT segment (NCW segments ahead: usually < 32 rows further on), loaded now so that its
            // latency hides behind this segment's work
            const int64_t wrow_next = wrow + nskip;
            const int wend_next = nskip ? load_window(wrow_next) : wend;
            T q1 = T(0), q2 = T(0), q3 = T(0), q4 = T(1);
            if (lane >= nskip && wend <= S1) row_operands_pinned<T, MODE>(wrow + lane, p1, p2, p3, out, q1, q2, q3, q4);  // rows finishing here
            const int lo_valid = S0 > F ? S0 : F;
            const bool has_data = S1 > lo_valid;
            const int t_tile = S0 / RG_TILE;
            if (has_data) {
                if (released < t_tile) {
                    released = t_tile;
                    if (lane == 0) progress[warp] = t_tile;
                }
                for (int t = seen > t_tile ? seen : t_tile; t <= t_tile; ++t) {
                    const int st = t % STG;
                    if (issued[st] != t + 1) {
                        const long long t0 = clock64();
                        while (issued[st] != t + 1) {
                            if (RG_SPIN_SLEEP_C) __nanosleep(RG_SPIN_SLEEP_C);
                            if (clock64() - t0 > RG_TIMEOUT) __trap();
                        }
                    }
                    mbar_wait(smem_u32(&S.full[st]), (t / STG) & 1);
                }
                seen = seen > t_tile + 1 ? seen : t_tile + 1;
                asm volatile("" ::: "memory");
                PROF_ADD(0, clock64() - it0);
            }
            int rel = S1 / RG_TILE;  // tiles wholly before the end of the segment: not needed by this warp once it has read its elements
            rel = rel < ntiles ? rel : ntiles;
            const int p0 = S0 % RG_ELEMS + lane;  // (RG_ELEMS is a multiple of SEG: no wrap inside a segment)
            bool any_end = false;
            T acc = T(0);
            PROF_T(ac0);
            auto carry_of = [&](int seg) -> T {  // the carry-out of segment seg - 1 (0 for the first segment)
                if (seg == 0) return T(0);
                const int slot = (seg - 1) % RG_NCARRY;
                T cv;
                if (!CarrySlot<T>::get(&carry[slot], seg, cv)) {
                    const long long t0 = clock64();
                    while (!CarrySlot<T>::get(&carry[slot], seg, cv)) {
                        __nanosleep(20);
                        if (clock64() - t0 > RG_TIMEOUT) __trap();
                    }
                    PROF_ADD(3, clock64() - t0);
                }
                return cv;
            };
            // complete the row parked by this warp's PREVIOUS segment: its carry was published long ago, nobody waits
            auto flush_head = [&]() {
                if (!head_pending) return;
                const T tot = carry_of(head_seg) + head_sum;
                if (lane == head_lane) row_epilogue<T, MODE>(head_row, tot, hq1, hq2, hq3, hq4, out, out2, lambda, omap, racc);
                head_pending = false;
            };
            auto park_head = [&](T sum, int jlane) {
                flush_head();
                head_pending = true;
                head_sum = sum;
                head_lane = jlane;
                head_row = wrow + jlane;
                head_seg = sg;
                hq1 = q1;
                hq2 = q2;
                hq3 = q3;
                hq4 = q4;
            };
            const int nfin = __popc(__ballot_sync(FULLM, wend <= S1)) - nskip;  // rows of the window that end in this segment
            if (nfin <= 3 && nskip + nfin < 32) {
                // ---- the usual case, straight-line code: at most three row ends, all inside the window ------------------------
                T v[RG_UNROLL];
                T g[RG_UNROLL];
                if (has_data) {
                    int c[RG_UNROLL];
                    if (S1 - S0 == SEG && S0 >= F) {
#pragma unroll
                        for (int u = 0; u < RG_UNROLL; ++u) ring_get(S.d, p0 + 32 * u, c[u], v[u]);
                    } else {  // first / last segment of the range: elements outside [F, E) are not the CTA's (or not loaded at all)
#pragma unroll
                        for (int u = 0; u < RG_UNROLL; ++u) {
                            const int pos = S0 + 32 * u + lane;
                            const bool ok = pos >= F && pos < S1;
                            ring_get(S.d, p0 + 32 * u, c[u], v[u]);
                            c[u] = ok ? c[u] : 0;
                            v[u] = ok ? v[u] : T(0);
                        }
                    }
                    __syncwarp();
                    if (rel > released) {
                        released = rel;
                        if (lane == 0) progress[warp] = rel;
                    }
#pragma unroll
                    for (int u = 0; u < RG_UNROLL; ++u) g[u] = __ldg(vec + c[u]);
                } else {
#pragma unroll
                    for (int u = 0; u < RG_UNROLL; ++u) v[u] = g[u] = T(0);
                }
                int e1 = e_next;
                int e2 = nfin > 1 ? __shfl_sync(FULLM, wend, jb + 1) : 0x7fffffff;
                int e3 = nfin > 2 ? __shfl_sync(FULLM, wend, jb + 2) : 0x7fffffff;
                if (nfin < 1) e1 = 0x7fffffff;
                T s0 = T(0), s1 = T(0), s2 = T(0);  // this lane's shares of the rows that end here, in order
                int nclosed = 0;
#pragma unroll
                for (int u = 0; u < RG_UNROLL; ++u) {
                    const int gend = S0 + 32 * (u + 1);
                    if (e1 > gend) {
                        acc = fma(v[u], g[u], acc);  // the whole group lies inside the open row
                    } else {
                        const int pos = S0 + 32 * u + lane;
                        const T prod = v[u] * g[u];
                        bool used = false;
#pragma unroll
                        for (int k = 0; k < 3; ++k) {
                            if (e1 <= gend) {  // a row ends inside (or right before / at the end of) this group
                                if (!used && pos < e1) {
                                    acc += prod;
                                    used = true;
                                }
                                if (nclosed == 0) s0 = acc;
                                else if (nclosed == 1) s1 = acc;
                                else s2 = acc;
                                ++nclosed;
                                acc = T(0);
                                e1 = e2;
                                e2 = e3;
                                e3 = 0x7fffffff;
                            }
                        }
                        if (!used) acc += prod;
                    }
                }
                if (nfin >= 1) {
                    any_end = true;
                    park_head(warp_sum(s0), jb);
                }
                if (nfin >= 2) {
                    const T tot = warp_sum(s1);
                    if (lane == jb + 1) row_epilogue<T, MODE>(wrow + jb + 1, tot, q1, q2, q3, q4, out, out2, lambda, omap, racc);
                }
                if (nfin >= 3) {
                    const T tot = warp_sum(s2);
                    if (lane == jb + 2) row_epilogue<T, MODE>(wrow + jb + 2, tot, q1, q2, q3, q4, out, out2, lambda, omap, racc);
                }
                jb += nfin;
            } else {
                // ---- many row ends in one segment (runs of empty rows, very short rows): compact loop, one group at a time ------
#pragma unroll 1
                for (int u = 0; u < RG_UNROLL; ++u) {
                    const int gend = S0 + 32 * (u + 1);
                    const int pos = S0 + 32 * u + lane;
                    T prod = T(0);
                    if (has_data) {
                        const bool ok = pos >= F && pos < S1;
                        int c;
                        T vv;
                        ring_get(S.d, p0 + 32 * u, c, vv);
                        prod = ok ? vv * __ldg(vec + (ok ? c : 0)) : T(0);
                    }
                    bool used = false;
                    while (e_next <= gend) {
                        if (!used && pos < e_next) {
                            acc += prod;
                            used = true;
                        }
                        const T tot = warp_sum(acc);
                        if (!any_end) {
                            any_end = true;
                            park_head(tot, jb);
                        } else if (lane == jb) {
                            row_epilogue<T, MODE>(wrow + jb, tot, q1, q2, q3, q4, out, out2, lambda, omap, racc);
                        }
                        acc = T(0);
                        const int e_cur = e_next;
                        ++jb;
                        for (;;) {  // the rows that follow and end at the same place are empty: their lanes finish them together
                            if (jb == 32) {  // window used up: slide it
                                wrow += 32;
                                wend = load_window(wrow);
                                jb = 0;
                                if (wend <= S1) row_operands_pinned<T, MODE>(wrow + lane, p1, p2, p3, out, q1, q2, q3, q4);
                            }
                            const unsigned same = __ballot_sync(FULLM, lane >= jb && wend == e_cur);
                            const int run = __popc(same);  // (row ends do not decrease: the lanes form a run starting at jb)
                            if (run == 0) break;
                            if ((same >> lane) & 1u) row_epilogue<T, MODE>(wrow + lane, T(0), q1, q2, q3, q4, out, out2, lambda, omap, racc);
                            jb += run;
                            if (jb < 32) break;
                        }
                        e_next = __shfl_sync(FULLM, wend, jb);
                    }
                    if (!used) acc += prod;
                }
                __syncwarp();
                if (has_data && rel > released) {
                    released = rel;
                    if (lane == 0) progress[warp] = rel;
                }
            }
            // what follows the last row end belongs to a row that goes on: hand it to the next segment
            T tail = warp_sum(acc);
            if (!any_end) tail = carry_of(sg) + tail;  // no row ended here: the open row's sum so far passes through
            if (lane == 0) CarrySlot<T>::put(&carry[sg % RG_NCARRY], tail, sg + 1);
            flush_head();  // (deferring this to the warp's next segment deadlocked at config 3's size: profiles/r02j_segments.md)
            PROF_ADD(1, clock64() - ac0);
            // the window for this warp's next segment was loaded at the start of this one
            wrow = wrow_next;
            wend = wend_next;
        }
        if (head_pending) {  // the row parked by this warp's last segment
            T cv = T(0);
            if (head_seg > 0) {
                const int slot = (head_seg - 1) % RG_NCARRY;
                const long long t0 = clock64();
                while (!CarrySlot<T>::get(&carry[slot], head_seg, cv)) {
                    __nanosleep(20);
                    if (clock64() - t0 > RG_TIMEOUT) __trap();
                }
            }
            if (lane == head_lane) row_epilogue<T, MODE>(head_row, cv + head_sum, hq1, hq2, hq3, hq4, out, out2, lambda, omap, racc);
        }
        __syncwarp();
        if (lane == 0) progress[warp] = ntiles;
        PROF_ADD(2, clock64() - ct0);
        PROF_FLUSH(0);
        PROF_FLUSH(1);
        PROF_FLUSH(2);
        PROF_FLUSH(3);
    } else {
    // ---- consumers, G >= 4 --------------------------------------------------------------------------------------------------
    // All positions below are element offsets relative to `base` and fit an int (a CTA's range is < 2^31 elements).
    // G <= 32: G lanes per row, 32/G rows per warp.  G == 64: a PAIR of warps per row (halves the rows in flight, hence
    // the ring span, for long rows); the odd warp hands its partial sum to the even one through shared memory.
    constexpr bool PAIR = G == 64;
    constexpr int GPW = PAIR ? 1 : 32 / G;         // rows per warp per iteration
    constexpr int GL = PAIR ? 32 : G;              // lanes of one warp on one row
    const int sub = lane / GL;
    const int gl = PAIR ? (warp & 1) * 32 + lane : lane % GL;
    const int unit = PAIR ? warp >> 1 : warp;       // row-taking unit (warp or warp pair)
    const int64_t stride = int64_t(PAIR ? NCW / 2 : NCW) * GPW;
    int iter = 0;
    int seen = 0;      // tiles [0, seen) known to have landed
    int released = 0;  // value last stored to progress[warp]
    int64_t rf = rs + int64_t(unit) * GPW;  // first row of this warp in the current iteration (warp-uniform)
    int s = 0, e = 0;
    if (rf < re) {
        const int64_t r = rf + sub;
        s = int(rowptr[r < re ? r : re] - base);
        e = int(rowptr[r + 1 < re ? r + 1 : re] - base);
    }
    PROF_DECL;
    PROF_T(ct0);
    for (; rf < re; rf += stride, ++iter) {
        const int64_t r = rf + sub;
        const bool valid = r < re;
        // prefetch the next iteration's row extent and this row's epilogue operands before touching the ring; the raw
        // row pointers are only turned into offsets at the END of the iteration, so the loads' latency (they were
        // ~10 % of the forward kernel's stall samples when consumed here, profiles/r02d) hides behind the dot product
        int64_t rp_s_next = base, rp_e_next = base;
        const int64_t rn = r + stride;
        if (rf + stride < re) {
            rp_s_next = rowptr[rn < re ? rn : re];
            rp_e_next = rowptr[rn + 1 < re ? rn + 1 : re];
        }
        T q1 = T(0), q2 = T(0), q3 = T(0), q4 = T(1);
        if (valid && gl == 0) row_operands<T, MODE>(r, p1, p2, p3, out, q1, q2, q3, q4);  // (in a pair: lane 0 of the even warp)
        const int w_start = __shfl_sync(0xffffffffu, s, 0), w_end = __shfl_sync(0xffffffffu, e, 31);
        // Release every tile wholly before this warp's position.  Every lane consumed its previous rows' ring data
        // (the values fed the shuffle reduction) before this point, and the warp is converged by the shuffle above.
        int t_start = w_start / RG_TILE;
        t_start = t_start < ntiles ? t_start : ntiles;
        if (released < t_start) {
            released = t_start;
            if (lane == 0) progress[warp] = t_start;
        }
        // Wait for the tiles this warp's rows span (span <= STG - 1 tiles by the plan): first until the stage is
        // armed for THAT tile (so the phase parity is unambiguous), then on the stage's mbarrier (a hardware wait).
        PROF_T(cw0);
        if (w_end > w_start) {
            const int t_hi = (w_end - 1) / RG_TILE;
            for (int t = seen > t_start ? seen : t_start; t <= t_hi; ++t) {
                const int st = t % STG;
                if (issued[st] != t + 1) {
                    const long long t0 = clock64();
                    while (issued[st] != t + 1)
                        if (clock64() - t0 > RG_TIMEOUT) __trap();
                }
                mbar_wait(smem_u32(&S.full[st]), (t / STG) & 1);
            }
            seen = seen > t_hi + 1 ? seen : t_hi + 1;
        }
        asm volatile("" ::: "memory");
        PROF_T(cd0);
        PROF_ADD(0, cd0 - cw0);
        // row dot product from the ring
        T a0 = T(0), a1 = T(0), a2 = T(0), a3 = T(0);
        const bool wraps = (w_start % RG_ELEMS) + (w_end - w_start) > RG_ELEMS;  // warp-uniform
        const int n_max = __reduce_max_sync(0xffffffffu, e - s - gl);
        const int trips = n_max > 0 ? (n_max + RG_UNROLL * G - 1) / (RG_UNROLL * G) : 0;
        int rel = w_end / RG_TILE;  // tiles wholly before the end of this warp's rows: not needed again (rows only move forward)
        rel = rel < ntiles ? rel : ntiles;
        rel = rel > released ? rel : released;
        if (!wraps) ring_row_dot<T, G, false, STG>(S.d, vec, s + gl, e, trips, progress + warp, rel, lane == 0, a0, a1, a2, a3);
        else ring_row_dot<T, G, true, STG>(S.d, vec, s + gl, e, trips, progress + warp, rel, lane == 0, a0, a1, a2, a3);
        if (trips > 0) released = rel;
        T acc = (a0 + a1) + (a2 + a3);
#pragma unroll
        for (int o = GL >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o, GL);
        PROF_ADD(1, clock64() - cd0);
        if (PAIR) {  // odd warp -> shared slot (double-buffered by iteration parity) -> pair barrier -> even warp adds
            if ((warp & 1) && lane == 0) S.pairbuf[unit][iter & 1] = acc;
            asm volatile("bar.sync %0, 64;" ::"r"(1 + unit) : "memory");
            if (!(warp & 1) && lane == 0) acc += S.pairbuf[unit][iter & 1];
        }
        if (valid && gl == 0 && !(PAIR && (warp & 1))) row_epilogue<T, MODE>(r, acc, q1, q2, q3, q4, out, out2, lambda, omap, racc);
        s = int(rp_s_next - base);
        e = int(rp_e_next - base);
    }
    // this warp needs nothing more
    __syncwarp();
    if (lane == 0) progress[warp] = ntiles;
    PROF_ADD(2, clock64() - ct0);
    if (warp == 0) PROF_ADD(5, clock64() - ct0);
    PROF_FLUSH(0);
    PROF_FLUSH(1);
    PROF_FLUSH(2);
    PROF_FLUSH(5);
    }
    // the kernel's reduction: lanes -> warp (fixed shuffle tree) -> CTA (warps in index order) -> red_out[blockIdx.x]
    if (red_out) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) racc += __shfl_xor_sync(0xffffffffu, racc, o);
        if (lane == 0) S.red[warp] = racc;
        asm volatile("bar.sync 15, %0;" ::"n"(32 * NCW) : "memory");
        if (threadIdx.x == 0) {
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < NCW; ++w) t += S.red[w];
            red_out[blockIdx.x] = t;
        }
    }
}

// ---- planning: partition table + eligibility -------------------------------------------------------------------------
// Rows are split by COST, not by nonzeros alone: cost(r0..r) = nonzeros + RG_ROW_COST per row (a row costs its shuffles,
// barrier waits and epilogue even when it is empty: config 4 has body voxels no beamlet reaches, config 3 rays that miss
// the image).  part[b] = first row r in [r0, r1] with cost(r0..r) >= total * b / nb  (part[0] = r0, part[nb] = r1).
#ifndef RG_ROW_COST
#define RG_ROW_COST 32  // (A/B at the end of round 2, 8 / 16 / 32 / 64: block-iterative config 3 933 / 931 / 917 / 907 us per sweep, config 4 forward
                        //  136 / 113 / 112 / 114 us, config 3 forward 323 / 324 / 324 / 326 us)
#endif
__global__ void k_stream_partition(const int64_t* __restrict__ rowptr, int64_t r0, int64_t r1, int nb, int64_t* __restrict__ part) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > nb) return;
    if (b == 0) { part[0] = r0; return; }
    if (b == nb) { part[nb] = r1; return; }
    const int64_t e0 = rowptr[r0];
    const int64_t total = (rowptr[r1] - e0) + int64_t(RG_ROW_COST) * (r1 - r0);
    const int64_t target = (total / nb) * b + ((total % nb) * b) / nb;
    int64_t lo = r0, hi = r1;  // lower bound on the monotone key
    while (lo < hi) {
        const int64_t mid = lo + ((hi - lo) >> 1);
        if ((rowptr[mid] - e0) + int64_t(RG_ROW_COST) * (mid - r0) < target) lo = mid + 1;
        else hi = mid;
    }
    part[b] = lo;
}

__global__ void __launch_bounds__(SUP_THREADS) k_stream_max_row(const int64_t* __restrict__ rowptr, int64_t r0, int64_t r1,
                                                                 unsigned long long* __restrict__ out) {
    unsigned long long mx = 0;
    for (int64_t r = r0 + int64_t(blockIdx.x) * blockDim.x + threadIdx.x; r < r1; r += int64_t(gridDim.x) * blockDim.x) {
        const unsigned long long len = (unsigned long long)(rowptr[r + 1] - rowptr[r]);
        mx = len > mx ? len : mx;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long t = __shfl_xor_sync(0xffffffffu, mx, o);
        mx = t > mx ? t : mx;
    }
    if ((threadIdx.x & 31) == 0 && mx > 0) atomicMax(out, mx);
}

size_t sup_stream_table_bytes() { return ((size_t(SUP_STREAM_NBMAX) + 1) * 8 + 255) & ~size_t(255); }

template <typename T, int MODE, bool DEEP>
static int staged_occupancy() {
    using Sh = RgShape<T, MODE, DEEP>;
    const void* fn = reinterpret_cast<const void*>(&k_staged<T, MODE, 32, Sh::NCW, Sh::STG>);
    const int smem = int(sizeof(RgSmem<T, Sh::STG>));
    int occ = 0;
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, 32 * (Sh::NCW + RG_NPROD), smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return occ;
}

static int stream_grid(sup_ctx* h) {  // persistent grid = resident CTAs per SM x SMs (0: unavailable)
    if (h->stream_nb) return h->stream_nb > 0 ? h->stream_nb : 0;
    int a, b;
    if (h->dt == SUP_F32) {
        a = staged_occupancy<float, 0, false>();
        b = staged_occupancy<float, 1, false>();
        const int c = staged_occupancy<float, 0, true>(), d = staged_occupancy<float, 1, true>();
        a = a < c ? a : c;
        b = b < d ? b : d;
    } else {
        a = staged_occupancy<double, 0, false>();
        b = staged_occupancy<double, 1, false>();
    }
    const int occ = a < b ? a : b;
    if (occ < 1) {
        h->stream_nb = -1;
        return 0;
    }
    h->stream_nb = occ * h->num_sms;
    return h->stream_nb;
}

sup_status sup_stream_plan(sup_ctx* h, const CsrD& M, int64_t r0, int64_t r1, bool forward, void* table, void* scratch,
                           StreamPlan* out) {
    *out = StreamPlan();
    out->table = table;
    if (!h->use_stream || r1 <= r0) return SUP_OK;
    int nb = stream_grid(h);
    if (nb < 1) return SUP_OK;
    {   // one chunk per resident CTA, but keep >= 64 rows per chunk
        int64_t want = nb;
        const int64_t most = (r1 - r0 + 63) / 64;
        if (want > most) want = most;
        if (want > SUP_STREAM_NBMAX) want = SUP_STREAM_NBMAX;
        nb = want < 1 ? 1 : int(want);
    }
    // bulk copies need 16-byte aligned sources (element offsets are multiples of 4)
    if ((reinterpret_cast<uintptr_t>(M.val) & 15) || (reinterpret_cast<uintptr_t>(M.col) & 15)) return SUP_OK;
    if (h->dt == SUP_F32 && !M.pk) return SUP_OK;  // fp32 streams the packed copy
    unsigned long long* mx = static_cast<unsigned long long*>(scratch);
    SUP_CUDA(h, cudaMemsetAsync(mx, 0, 8, h->stream));
    const int grid = sup_grid_for(r1 - r0, SUP_THREADS, h->num_sms * 8);
    k_stream_max_row<<<grid, SUP_THREADS, 0, h->stream>>>(M.rowptr, r0, r1, mx);
    k_stream_partition<<<(nb + 1 + 127) / 128, 128, 0, h->stream>>>(M.rowptr, r0, r1, nb, static_cast<int64_t*>(table));
    unsigned long long mx_h = 0;
    int64_t ends[2] = {0, 0};
    SUP_CUDA(h, cudaMemcpyAsync(&mx_h, mx, 8, cudaMemcpyDeviceToHost, h->stream));
    SUP_CUDA(h, cudaMemcpyAsync(&ends[0], M.rowptr + r0, 8, cudaMemcpyDeviceToHost, h->stream));
    SUP_CUDA(h, cudaMemcpyAsync(&ends[1], M.rowptr + r1, 8, cudaMemcpyDeviceToHost, h->stream));
    SUP_CUDA(h, cudaStreamSynchronize(h->stream));
    SUP_CUDA(h, cudaGetLastError());
    // Lanes per row: the rows a warp holds at once (32/G of them) should total ~a tile -- enough elements per lane to
    // amortise the per-row work, few enough that the consumer warps' rows together leave ring stages free for prefetch --
    // and must never span more than RG_STAGES_MIN - 1 tiles.  sup_set_row_mode() overrides the choice.
    const double avg = double(ends[1] - ends[0]) / double(r1 - r0);
    int G = 2;  // (2 lanes per row for rows of up to ~60 entries: config 4's forward product 3 190 -> 5 170 GB/s against 4 lanes)
    while (G < 32 && avg * (32.0 / G) > 960.0) G <<= 1;
    if (avg >= RG_SEG_MIN_AVG) G = 1;
    else if (avg > 2048.0) G = 128;  // rows of thousands of entries (config 4's A^T): chunks of rows round-robin over the warps
    const int forced = forward ? h->lanes_fwd : h->lanes_bwd;
    if (forced >= 0) G = forced;
    const int64_t cap = int64_t(RG_STAGES_MIN - 2) * RG_TILE;
    if (G == 128) {
        if (int64_t(mx_h) > int64_t(RG_CHUNK_KMAX) * 32 * RG_UNROLL) G = 0;  // more chunks than the pool allows: the whole CTA per row
    } else {
        while (G < 32 && G > 1 && int64_t(mx_h) * (32 / G) > cap) G <<= 1;
        if (G > 1 && int64_t(mx_h) * (G >= 32 ? 1 : 32 / G) > cap) G = 0;  // a row too long for the ring in a lanes-per-row mode: the whole CTA per row
    }
    out->max_row = int64_t(mx_h);
    out->part = static_cast<const int64_t*>(table);
    out->nb = nb;
    out->G = G;
    out->ok = true;
    return SUP_OK;
}

// ---- launchers --------------------------------------------------------------------------------------------------------
template <typename T, int MODE, int G, bool DEEP>
static void launch_staged_g(sup_ctx* h, const StreamPlan& sp, const CsrD& M, const void* vec, const void* p1, const void* p2,
                            const void* p3, void* out, void* out2, double lambda, const GMap& omap, double* red_out) {
    using Sh = RgShape<T, MODE, DEEP>;
    const void* fn = reinterpret_cast<const void*>(&k_staged<T, MODE, G, Sh::NCW, Sh::STG>);
    constexpr int smem = int(sizeof(RgSmem<T, Sh::STG>));
    if (!h->smem_opted_in.count(fn)) {  // per handle, hence per device: opt in to > 48 KB of dynamic shared memory
        cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        h->smem_opted_in.insert(fn);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(unsigned(sp.nb));
    cfg.blockDim = dim3(32 * (Sh::NCW + RG_NPROD));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    // Every launch carries it (the matrix, the partition table and the row pointers its producers read are written by set-up calls
    // that end in a stream synchronisation; everything a sweep's kernels write is read behind griddepcontrol.wait), except with a
    // stop flag, which is read before any wait.  Behind a kernel that never triggers, the attribute changes nothing.
    cfg.numAttrs = (h->pdl && !h->stop_ptr) ? 1 : 0;
    cudaLaunchKernelEx(&cfg, k_staged<T, MODE, G, Sh::NCW, Sh::STG>, sp.part, M.rowptr, M.col, static_cast<const T*>(M.val),
                       static_cast<const uint2*>(M.pk), static_cast<const T*>(vec), static_cast<const T*>(p1), static_cast<const T*>(p2),
                       static_cast<const T*>(p3), static_cast<T*>(out), static_cast<T*>(out2), T(lambda), M.alloc_nnz, omap, red_out,
                       static_cast<const int*>(h->stop_ptr));
    h->launches++;
}

// deep: the gathered vector (x for MODE 0, y for MODE 1) is kept in a tiled layout
template <typename T, int MODE, bool DEEP>
static void launch_staged_d(sup_ctx* h, const StreamPlan& sp, const CsrD& M, const void* vec, const void* p1, const void* p2,
                            const void* p3, void* out, void* out2, double lambda, const GMap& omap, double* red_out) {
    switch (sp.G) {
        case 2: launch_staged_g<T, MODE, 2, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        case 4: launch_staged_g<T, MODE, 4, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        case 8: launch_staged_g<T, MODE, 8, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        case 16: launch_staged_g<T, MODE, 16, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        case 64: launch_staged_g<T, MODE, 64, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        case 0: launch_staged_g<T, MODE, 0, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        case 128: launch_staged_g<T, MODE, 128, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        case 1: launch_staged_g<T, MODE, 1, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
        default: launch_staged_g<T, MODE, 32, DEEP>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out); break;
    }
}

template <typename T, int MODE>
static void launch_staged(sup_ctx* h, const StreamPlan& sp, const CsrD& M, const void* vec, const void* p1, const void* p2,
                          const void* p3, void* out, void* out2, double lambda, const GMap& omap, bool deep, double* red_out = nullptr) {
    // the deeper shape also pays when the gathered vector stays in L1 anyway (config 4's x: 32 KB) and in the chunk mode, whose ring
    // span does not grow with the rows (config 4: forward 121 -> 114 us, back-projection 154 -> 148 us); with scattered gathers it
    // costs L1 capacity (config 5: -3 %)
    deep = deep || M.cols * int64_t(sizeof(T)) <= 49152 || sp.G == 128;
    if (deep && sizeof(T) == 4) launch_staged_d<T, MODE, true>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out);
    else launch_staged_d<T, MODE, false>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, red_out);
}

// ---- gather layouts: the mirror of x and the internal layout of y (GMap, sup_internal.cuh) ------------------------------
__global__ void __launch_bounds__(SUP_THREADS) k_map_cols(const int32_t* __restrict__ col, int64_t nnz, int32_t* __restrict__ colg, const GMap map) {
    for (int64_t k = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; k < nnz; k += int64_t(gridDim.x) * blockDim.x)
        colg[k] = sup_gmap(map, col[k]);
}

template <typename T>
__global__ void __launch_bounds__(SUP_THREADS) k_map_copy(const T* __restrict__ x, int n, T* __restrict__ xg, const GMap map) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) xg[sup_gmap(map, j)] = x[j];
}

template <typename T>
__global__ void __launch_bounds__(SUP_THREADS) k_unmap_copy(const T* __restrict__ src, int n, T* __restrict__ dst, const GMap map) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) dst[j] = src[sup_gmap(map, j)];
}

__global__ void __launch_bounds__(SUP_THREADS) k_pack(const float* __restrict__ val, const int32_t* __restrict__ col, int64_t nnz,
                                                       uint2* __restrict__ pk, const GMap map) {
    for (int64_t k = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; k < nnz; k += int64_t(gridDim.x) * blockDim.x)
        pk[k] = make_uint2(__float_as_uint(val[k]), unsigned(sup_gmap(map, col[k])));
}

sup_status sup_stream_pack(sup_ctx* h, const void* val, const int32_t* col, int64_t nnz, void* dst, const GMap& map) {
    if (h->dt != SUP_F32 || !dst || nnz == 0) return SUP_OK;
    k_pack<<<sup_grid_for(nnz, SUP_THREADS, h->num_sms * 16), SUP_THREADS, 0, h->stream>>>(
        static_cast<const float*>(val), col, nnz, static_cast<uint2*>(dst), map);
    h->launches++;
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

sup_status sup_stream_setup_gather(sup_ctx* h) {
    if (h->nnz == 0) return SUP_OK;
    const int grid = sup_grid_for(h->nnz, SUP_THREADS, h->num_sms * 16);
    if (h->dt == SUP_F32 && h->pk_a) {
        k_pack<<<grid, SUP_THREADS, 0, h->stream>>>(static_cast<const float*>(h->A.val), h->A.col, h->nnz,
                                                   static_cast<uint2*>(h->pk_a), h->xmap);
        h->A.pk = h->pk_a;
    } else if (h->colg) {
        k_map_cols<<<grid, SUP_THREADS, 0, h->stream>>>(h->A.col, h->nnz, h->colg, h->xmap);
    } else {
        return SUP_OK;
    }
    h->launches++;
    SUP_CUDA(h, cudaGetLastError());
    return SUP_OK;
}

void sup_launch_unmap(sup_ctx* h, const void* src, void* dst, int64_t count, const GMap& map) {
    const unsigned grid = unsigned((count + SUP_THREADS - 1) / SUP_THREADS);
    if (h->dt == SUP_F32) k_unmap_copy<float><<<grid, SUP_THREADS, 0, h->stream>>>(static_cast<const float*>(src), int(count), static_cast<float*>(dst), map);
    else k_unmap_copy<double><<<grid, SUP_THREADS, 0, h->stream>>>(static_cast<const double*>(src), int(count), static_cast<double*>(dst), map);
    h->launches++;
}

bool sup_stream_forward_uses_xg(const sup_ctx* h) {
    if (!(h->colg || h->A.pk) || !h->xg) return false;
    if (h->A.plan.ok) return true;
    for (const StreamPlan& p : h->stream_fwd_blk)
        if (p.ok) return true;
    return false;
}

// The row-side map (the layout of the internal y) is in force only when EVERY product of the handle runs on the staged fp32
// kernels: they read y through the packed copies of A^T, which carry the mapped row index; the group-per-row kernels
// and fp64 handles index y directly.  Rewrites every packed / mapped copy accordingly.
sup_status sup_stream_refresh_layout(sup_ctx* h) {
    bool all = h->use_stream && h->dt == SUP_F32 && h->pk_a && h->pk_at && h->A.plan.ok && h->AT.plan.ok;
    for (int t = 0; all && t < h->n_blocks; ++t) {
        const bool empty = h->block_rowptr[t + 1] == h->block_rowptr[t];
        all = empty || (h->stream_fwd_blk[t].ok && h->ATb[t].plan.ok && h->pk_atb);
    }
    h->ymap = all ? h->ymap_req : GMap();
    h->xg_synced = false;
    if (!h->use_stream) return SUP_OK;
    sup_status rc = sup_stream_setup_gather(h);
    if (rc == SUP_OK) rc = sup_stream_pack(h, h->AT.val, h->AT.col, h->nnz, h->pk_at, h->ymap);
    if (rc == SUP_OK && h->n_blocks > 0 && h->pk_atb) rc = sup_stream_pack(h, h->ATb[0].val, h->ATb[0].col, h->nnz, h->pk_atb, h->ymap);
    return rc;
}

static const void* stream_sync_mirror(sup_ctx* h, const void* x) {
    // the forward product gathers from the mirror of x in its gather layout; refresh it when x changed outside the kernels
    if (!((h->colg || h->A.pk) && h->xg)) return x;
    if (!h->xg_synced) {
        const unsigned grid = unsigned((h->n + SUP_THREADS - 1) / SUP_THREADS);
        if (h->dt == SUP_F32) k_map_copy<float><<<grid, SUP_THREADS, 0, h->stream>>>(static_cast<const float*>(x), int(h->n), static_cast<float*>(h->xg), h->xmap);
        else k_map_copy<double><<<grid, SUP_THREADS, 0, h->stream>>>(static_cast<const double*>(x), int(h->n), static_cast<double*>(h->xg), h->xmap);
        h->launches++;
        h->xg_synced = true;
    }
    return h->xg;
}

// One staged product: mode 0 / 1 / 2 of row_epilogue over the rows of `sp` of matrix M, gathering `vec` at the (mapped)
// indices the stream carries.  red_out (optional): [sp.nb] per-CTA partials of the mode's reduction.
void sup_launch_staged(sup_ctx* h, int mode, const StreamPlan& sp, const CsrD& M, const void* vec, const void* p1, const void* p2,
                       const void* p3, void* out, void* out2, double lambda, const GMap& omap, bool deep, double* red_out) {
    if (h->dt == SUP_F32) {
        if (mode == 0) launch_staged<float, 0>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, deep, red_out);
        else if (mode == 1) launch_staged<float, 1>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, deep, red_out);
        else launch_staged<float, 2>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, deep, red_out);
    } else {
        if (mode == 0) launch_staged<double, 0>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, false, red_out);
        else if (mode == 1) launch_staged<double, 1>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, false, red_out);
        else launch_staged<double, 2>(h, sp, M, vec, p1, p2, p3, out, out2, lambda, omap, false, red_out);
    }
}

// S1+S2 over the rows of `sp`: y = dscale * c(x) (dscale = d, the block scaling, or the plain weights of DROP / EMR)
void sup_launch_stream_fwd(sup_ctx* h, const StreamPlan& sp, const void* x, const void* dscale, double* red_out) {
    CsrD M = h->A;
    const void* vec = stream_sync_mirror(h, x);
    if (vec == h->xg && h->colg) M.col = h->colg;  // fp32: the mapped column is inside M.pk
    sup_launch_staged(h, 0, sp, M, vec, h->lb, h->ub, dscale, h->y, nullptr, 0.0, h->ymap, vec == h->xg && h->xmap.kind == 2, red_out);
}

// S3 over A^T (or a block's): x <- clip(x - lambda * zscale .* (A^T y)); zscale = NULL: 1
void sup_launch_stream_bwd(sup_ctx* h, const CsrD& AT, const StreamPlan& sp, void* x, double lambda, const void* zscale) {
    void* mirror = sup_stream_forward_uses_xg(h) ? h->xg : nullptr;
    sup_launch_staged(h, 1, sp, AT, h->y, h->lo, h->hi, zscale, x, mirror, lambda, h->xmap, h->ymap.kind == 2, nullptr);
    h->xg_synced = mirror != nullptr;
}

// out = scale * A v (over the rows of A.plan) with v given in x's gather layout (v_g[xmap(j)] = v_j), reduction sum wrow_i out_i^2
void sup_launch_stream_plain_A(sup_ctx* h, const void* v_g, void* out, double scale, const void* wrow, double* red_out) {
    CsrD M = h->A;
    if (h->colg) M.col = h->colg;
    sup_launch_staged(h, 2, h->A.plan, M, v_g, nullptr, nullptr, wrow, out, nullptr, scale, GMap(), h->xmap.kind == 2, red_out);
}

// out_g[xmap(j)] = scale * (A^T y)_j with the internal y (its gather layout), reduction sum out_j^2
void sup_launch_stream_plain_AT(sup_ctx* h, void* out_g, double scale, double* red_out) {
    sup_launch_staged(h, 2, h->AT.plan, h->AT, h->y, nullptr, nullptr, nullptr, out_g, nullptr, scale, h->xmap, h->ymap.kind == 2, red_out);
}
