"""Workload recipes for BASELINE.json configs 1-5 (see gen/__init__.py for the role of this package).

All randomness comes from numpy PCG64 streams seeded with SEED0 + config index (configs 1-4) or from
a pure-integer counter hash (config 5, so that a device generator can reproduce it bit for bit).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

SEED0 = 20260627
_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "_gen.c")
_LIB = os.path.join(_HERE, "_gen.so")
_lib = None

_i64p = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")


def build_native(force: bool = False) -> str:
    """Compile gen/_gen.c -> gen/_gen.so (gcc -O2 -fopenmp) if missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _native():
    global _lib
    if _lib is None:
        build_native()
        L = ctypes.CDLL(_LIB)
        c_int, c_dbl, c_i64 = ctypes.c_int, ctypes.c_double, ctypes.c_int64
        L.ct_count.argtypes = [c_int, c_int, c_dbl, c_int, c_int, _i64p]
        L.ct_fill.argtypes = [c_int, c_int, c_dbl, c_int, c_int, _i64p, _i32p, _f32p]
        L.seg_count.argtypes = [c_i64, _f64p, c_int, c_int, _i64p]
        L.seg_fill.argtypes = [c_i64, _f64p, c_int, c_int, _i64p, _i32p, _f32p]
        imrt_common = [c_int, c_int, c_int, c_dbl, c_int, _f64p, c_int, c_dbl, c_dbl, c_dbl, c_dbl, c_dbl, c_i64, _i64p]
        L.imrt_colmax.argtypes = imrt_common + [_f64p]
        L.imrt_rows.argtypes = imrt_common + [_f64p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        for f in (L.ct_count, L.ct_fill, L.seg_count, L.seg_fill, L.imrt_colmax, L.imrt_rows):
            f.restype = None
        _lib = L
    return _lib


@dataclass
class Problem:
    """One hyperslab + box feasibility problem with its superiorization parameters (all arrays fp32/int)."""

    name: str
    m: int
    n: int
    rowptr: np.ndarray  # int64 [m+1]
    col: np.ndarray  # int32 [nnz], sorted & distinct within a row
    val: np.ndarray  # float32 [nnz]
    lb: np.ndarray  # float32 [m]  (-inf allowed)
    ub: np.ndarray  # float32 [m]  (+inf allowed)
    lo: np.ndarray  # float32 [n]
    hi: np.ndarray  # float32 [n]
    x0: np.ndarray  # float32 [n]
    objective: Optional[str] = None  # 'tv2d' | 'tv1d' | 'dose' | None
    shape: Optional[tuple] = None  # image shape for TV
    n_sweeps: int = 10
    N: int = 0
    beta0: float = 1.0
    a: float = 0.99
    lam: float = 1.0
    weights: Optional[np.ndarray] = None
    x_true: Optional[np.ndarray] = None
    dose: Optional[tuple] = None  # (rowptr, col, val, m_d) of D_body
    block_rowptr: Optional[np.ndarray] = None  # int64 [B+1], rows are block-contiguous
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.rowptr[-1])

    def scipy(self):
        import scipy.sparse as sp

        ip = self.rowptr.astype(np.int32) if self.nnz < 2**31 else self.rowptr
        return sp.csr_matrix((self.val.astype(np.float64), self.col, ip), shape=(self.m, self.n))


# ----------------------------------------------------------------------------------------------
# matrices
# ----------------------------------------------------------------------------------------------
def _finish(counts, fill):
    rowptr = np.zeros(counts.size + 1, np.int64)
    np.cumsum(counts, out=rowptr[1:])
    nnz = int(rowptr[-1])
    col = np.empty(nnz, np.int32)
    val = np.empty(nnz, np.float32)
    fill(rowptr, col, val)
    return rowptr, col, val


def ct_matrix(n_pix: int, n_angles: int, n_bins: int, spacing: float = 1.0):
    """Parallel-beam CT system matrix: exact ray/pixel intersection lengths on an n_pix x n_pix grid of unit
    pixels centred at the origin; row q*n_bins+p is the line x cos(th_q) + y sin(th_q) = (p-(n_bins-1)/2)*spacing,
    th_q = q*pi/n_angles; pixel (i,j) (i along y, j along x) has index i*n_pix+j."""
    L = _native()
    counts = np.zeros(n_angles * n_bins, np.int64)
    L.ct_count(n_angles, n_bins, spacing, n_pix, n_pix, counts)
    return _finish(counts, lambda rp, c, v: L.ct_fill(n_angles, n_bins, spacing, n_pix, n_pix, rp, c, v))


def segment_matrix(segments: np.ndarray, nx: int, ny: int):
    """Path lengths of straight segments (xs,ys)->(xr,yr) through unit cells of the grid [0,nx]x[0,ny]."""
    L = _native()
    seg = np.ascontiguousarray(segments, np.float64)
    m = seg.shape[0]
    counts = np.zeros(m, np.int64)
    L.seg_count(m, seg, nx, ny, counts)
    return _finish(counts, lambda rp, c, v: L.seg_fill(m, seg, nx, ny, rp, c, v))


def imrt_matrix(grid, h, phis, nb, bs, mu, sigma, depth0, trunc, vox):
    """Pencil-beam dose-influence rows for the voxels `vox` (linear indices (z*gy+y)*gx+x)."""
    L = _native()
    gx, gy, gz = grid
    phis = np.ascontiguousarray(phis, np.float64)
    vox = np.ascontiguousarray(vox, np.int64)
    colmax = np.zeros(phis.size * nb * nb, np.float64)
    args = (gx, gy, gz, float(h), phis.size, phis, nb, float(bs), float(mu), float(sigma), float(depth0), float(trunc), vox.size, vox)
    L.imrt_colmax(*args, colmax)
    counts = np.zeros(vox.size, np.int64)
    L.imrt_rows(*args, colmax, None, counts.ctypes.data, None, None)

    def fill(rp, c, v):
        L.imrt_rows(*args, colmax, rp.ctypes.data, None, c.ctypes.data, v.ctypes.data)

    return _finish(counts, fill)


# ----------------------------------------------------------------------------------------------
# phantoms
# ----------------------------------------------------------------------------------------------
def _ellipse_phantom(rng, n_pix, n_ell):
    """Sum of n_ell random ellipses on [-1,1]^2 sampled at pixel centres, clipped to [0,1]."""
    c = (np.arange(n_pix) + 0.5) / n_pix * 2.0 - 1.0
    X, Y = np.meshgrid(c, c)  # X varies along j (fast index), Y along i
    img = np.zeros((n_pix, n_pix))
    for _ in range(n_ell):
        cx, cy = rng.uniform(-0.5, 0.5, 2)
        ax, ay = rng.uniform(0.1, 0.4, 2)
        th = rng.uniform(0.0, np.pi)
        amp = rng.uniform(0.1, 0.5)
        xr = (X - cx) * np.cos(th) + (Y - cy) * np.sin(th)
        yr = -(X - cx) * np.sin(th) + (Y - cy) * np.cos(th)
        img += amp * ((xr / ax) ** 2 + (yr / ay) ** 2 <= 1.0)
    return np.clip(img, 0.0, 1.0).ravel()


def _f32_down(x):
    y = x.astype(np.float32)
    bad = y.astype(np.float64) > x
    y[bad] = np.nextafter(y[bad], np.float32(-np.inf))
    return y


def _f32_up(x):
    y = x.astype(np.float32)
    bad = y.astype(np.float64) < x
    y[bad] = np.nextafter(y[bad], np.float32(np.inf))
    return y


# ----------------------------------------------------------------------------------------------
# configs
# ----------------------------------------------------------------------------------------------
def config1_tiny_ct(n_pix=64, n_angles=90, n_bins=91, n_sweeps=50, N=5, seed=SEED0 + 1) -> Problem:
    """BASELINE.json configs[0]: tiny parallel-beam CT, Gaussian noise 1 % of max(b), bounds b +/- 2 sigma, box [0,1]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    rowptr, col, val = ct_matrix(n_pix, n_angles, n_bins)
    n, m = n_pix * n_pix, n_angles * n_bins
    x_true = _ellipse_phantom(rng, n_pix, 6).astype(np.float32)
    P = Problem("cfg1_tiny_ct", m, n, rowptr, col, val, None, None, None, None, None)
    b = P.scipy() @ x_true.astype(np.float64)
    sigma = 0.01 * b.max()
    b = b + rng.normal(0.0, sigma, m)
    P.lb, P.ub = (b - 2 * sigma).astype(np.float32), (b + 2 * sigma).astype(np.float32)
    P.lo, P.hi = np.zeros(n, np.float32), np.ones(n, np.float32)
    P.x0 = np.zeros(n, np.float32)
    P.x_true = x_true
    P.objective, P.shape = "tv2d", (n_pix, n_pix)
    P.n_sweeps, P.N, P.beta0, P.a, P.lam = n_sweeps, N, 1.0, 0.99, 1.0
    P.meta = dict(sigma=float(sigma), n_angles=n_angles, n_bins=n_bins)
    return P


def config2_crosswell(n_grid=128, n_src=64, n_rcv=64, n_sweeps=200, N=10, seed=SEED0 + 2) -> Problem:
    """BASELINE.json configs[1]: crosswell straight-ray travel-time tomography, noise 0.5 %, box [0.1,1.0]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    step = n_grid / n_src
    ys = (np.arange(n_src) + 0.5) * step
    yr = (np.arange(n_rcv) + 0.5) * (n_grid / n_rcv)
    seg = np.empty((n_src * n_rcv, 4))
    seg[:, 0] = 0.0
    seg[:, 1] = np.repeat(ys, n_rcv)
    seg[:, 2] = float(n_grid)
    seg[:, 3] = np.tile(yr, n_src)
    rowptr, col, val = segment_matrix(seg, n_grid, n_grid)
    n, m = n_grid * n_grid, n_src * n_rcv
    # four horizontal layers 0.2..0.5 (top to bottom), two Gaussian anomalies of +/-15 %
    ci = (np.arange(n_grid) + 0.5)
    Xc, Yc = np.meshgrid(ci, ci)
    layer = np.minimum((Yc / (n_grid / 4)).astype(int), 3)
    s_true = 0.2 + 0.1 * layer
    for sign in (+1.0, -1.0):
        cx, cy = rng.uniform(n_grid / 4, 3 * n_grid / 4, 2)
        s_true = s_true * (1.0 + sign * 0.15 * np.exp(-((Xc - cx) ** 2 + (Yc - cy) ** 2) / (2 * (n_grid / 16) ** 2)))
    s_true = s_true.ravel().astype(np.float32)
    P = Problem("cfg2_crosswell", m, n, rowptr, col, val, None, None, None, None, None)
    t = P.scipy() @ s_true.astype(np.float64)
    sigma = 0.005 * t.max()
    t = t + rng.normal(0.0, sigma, m)
    P.lb, P.ub = (t - 2 * sigma).astype(np.float32), (t + 2 * sigma).astype(np.float32)
    P.lo, P.hi = np.full(n, 0.1, np.float32), np.full(n, 1.0, np.float32)
    P.x0 = np.full(n, 0.1, np.float32)
    P.x_true = s_true
    P.objective, P.shape = "tv2d", (n_grid, n_grid)
    P.n_sweeps, P.N, P.beta0, P.a, P.lam = n_sweeps, N, 1.0, 0.995, 1.0
    P.meta = dict(sigma=float(sigma), segments=seg)
    return P


def config3_lowdose_ct(n_pix=512, n_angles=720, n_bins=729, n_sweeps=100, N=5, seed=SEED0 + 3, I0=1e4) -> Problem:
    """BASELINE.json configs[2]: low-dose CT with Poisson transmission noise; bounds +/- 2 local sigma; box [0,inf)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    rowptr, col, val = ct_matrix(n_pix, n_angles, n_bins)
    n, m = n_pix * n_pix, n_angles * n_bins
    x_true = _ellipse_phantom(rng, n_pix, 12)
    P = Problem("cfg3_lowdose_ct", m, n, rowptr, col, val, None, None, None, None, None)
    A = P.scipy()
    p = A @ x_true
    x_true = (x_true * (4.0 / p.max())).astype(np.float32)  # densest ray has line integral 4.0
    p = A @ x_true.astype(np.float64)
    del A
    counts = rng.poisson(I0 * np.exp(-p)).astype(np.float64)
    counts = np.maximum(counts, 1.0)
    p_hat = np.log(I0 / counts)
    sig = 1.0 / np.sqrt(counts)  # delta method: std of ln(I0/I)
    P.lb, P.ub = (p_hat - 2 * sig).astype(np.float32), (p_hat + 2 * sig).astype(np.float32)
    P.lo, P.hi = np.zeros(n, np.float32), np.full(n, np.inf, np.float32)
    P.x0 = np.zeros(n, np.float32)
    P.x_true = x_true
    P.objective, P.shape = "tv2d", (n_pix, n_pix)
    P.n_sweeps, P.N, P.beta0, P.a, P.lam = n_sweeps, N, 1.0, 0.99, 1.0
    P.meta = dict(n_angles=n_angles, n_bins=n_bins, I0=I0)
    return P


def interleaved_angle_blocks(P: Problem, n_blocks: int) -> Problem:
    """Permute the rows of a CT problem so that block t holds the angles q = t (mod n_blocks), contiguously
    (reading A-14).  Returns a new Problem with block_rowptr set."""
    na, nb = P.meta["n_angles"], P.meta["n_bins"]
    q = np.arange(na)
    order_q = np.concatenate([q[q % n_blocks == t] for t in range(n_blocks)])
    perm = (order_q[:, None] * nb + np.arange(nb)[None, :]).ravel()
    counts = np.diff(P.rowptr)[perm]
    rowptr = np.zeros(P.m + 1, np.int64)
    np.cumsum(counts, out=rowptr[1:])
    # gather entries row by row (vectorised through a repeat/arange trick)
    starts = P.rowptr[:-1][perm]
    idx = np.repeat(starts - rowptr[:-1], counts) + np.arange(rowptr[-1], dtype=np.int64)
    blk = np.array([np.sum(q % n_blocks < t) for t in range(n_blocks + 1)], np.int64) * nb
    Q = Problem(P.name + f"_bip{n_blocks}", P.m, P.n, rowptr, P.col[idx], P.val[idx], P.lb[perm], P.ub[perm], P.lo, P.hi, P.x0,
                P.objective, P.shape, P.n_sweeps, P.N, P.beta0, P.a, P.lam, None, P.x_true, None, blk, dict(P.meta, row_perm=perm))
    return Q


def config4_imrt(scale=1.0, infeasible=False, n_sweeps=300, N=3, seed=SEED0 + 4) -> Problem:
    """BASELINE.json configs[3]: synthetic IMRT.  scale < 1 shrinks the voxel grid and beamlet count
    (same physical extent, coarser sampling) for tests; scale = 1 is the full 160x160x100 / 8000-beamlet case."""
    rng = np.random.Generator(np.random.PCG64(seed))
    gx, gy, gz = (max(8, int(round(160 * scale))), max(8, int(round(160 * scale))), max(6, int(round(100 * scale))))
    h = 3.0 * 160 / gx
    nb = max(4, int(round(40 * scale)))
    bs = 5.0 * 40 / nb
    sigma = 4.0 * max(1.0, bs / 5.0)  # keep the lateral profile resolved on coarse test grids
    phis = np.deg2rad([0.0, 72.0, 144.0, 216.0, 288.0])
    X = (np.arange(gx) - 0.5 * (gx - 1)) * h
    Y = (np.arange(gy) - 0.5 * (gy - 1)) * h
    Z = (np.arange(gz) - 0.5 * (gz - 1)) * h  # isotropic voxels (the C generator assumes one spacing)
    Zg, Yg, Xg = np.meshgrid(Z, Y, X, indexing="ij")
    body = (Xg / 240.0) ** 2 + (Yg / 240.0) ** 2 + (Zg / 150.0) ** 2 <= 1.0
    r_ptv, r1, r2 = 30.0, 20.0, 15.0
    # the infeasible variant overlaps OAR1 and the PTV by 5 mm (BASELINE.json); on the coarse test grids (scale < 1, voxels
    # up to 20 mm) by at least 1.6 voxels, so that some voxel centres do fall in both structures
    d1 = (r_ptv + r1 - max(5.0, 1.6 * h)) if infeasible else 65.0
    d2 = 60.0
    while True:
        a1, a2 = rng.uniform(0, 2 * np.pi, 2)
        c1 = np.array([d1 * np.cos(a1), d1 * np.sin(a1)])
        c2 = np.array([d2 * np.cos(a2), d2 * np.sin(a2)])
        if np.linalg.norm(c1 - c2) > r1 + r2 + 1.0:
            break
    ptv = Xg**2 + Yg**2 + Zg**2 <= r_ptv**2
    oar1 = (Xg - c1[0]) ** 2 + (Yg - c1[1]) ** 2 + Zg**2 <= r1**2
    oar2 = (Xg - c2[0]) ** 2 + (Yg - c2[1]) ** 2 + Zg**2 <= r2**2
    vox = np.flatnonzero(body.ravel()).astype(np.int64)
    rowptr, col, val = imrt_matrix((gx, gy, gz), h, phis, nb, bs, 0.005, sigma, 240.0, 1e-3, vox)
    m_d, n = vox.size, phis.size * nb * nb
    f = lambda mask: mask.ravel()[vox]
    is_ptv, is_o1, is_o2 = f(ptv), f(oar1), f(oar2)
    lb = np.full(m_d, -np.inf, np.float32)
    ub = np.full(m_d, 66.0, np.float32)
    ub[is_o2] = 30.0
    ub[is_o1] = 20.0
    lb[is_ptv], ub[is_ptv] = 57.0, 64.2
    dose = (rowptr, col, val, m_d)
    if infeasible:
        dup = np.flatnonzero(is_ptv & is_o1)  # voxels in PTV and OAR1 get a second row carrying the OAR bound
        counts = np.diff(rowptr)
        extra_counts = counts[dup]
        rp2 = np.zeros(m_d + dup.size + 1, np.int64)
        np.cumsum(np.concatenate([counts, extra_counts]), out=rp2[1:])
        idx = np.repeat(rowptr[:-1][dup] - rp2[m_d:-1], extra_counts) + np.arange(rp2[m_d], rp2[-1], dtype=np.int64)
        col2, val2 = np.concatenate([col, col[idx]]), np.concatenate([val, val[idx]])
        lb = np.concatenate([lb, np.full(dup.size, -np.inf, np.float32)])
        ub = np.concatenate([ub, np.full(dup.size, 20.0, np.float32)])
        A = (rp2, col2, val2)
    else:
        A = (rowptr, col, val)
    m = A[0].size - 1
    P = Problem("cfg4_imrt" + ("_infeasible" if infeasible else ""), m, n, A[0], A[1], A[2], lb, ub,
                np.zeros(n, np.float32), np.full(n, np.inf, np.float32), np.zeros(n, np.float32))
    P.objective, P.dose = "dose", dose
    P.n_sweeps, P.N, P.beta0, P.a, P.lam = n_sweeps, N, 1.0, 0.99, 1.0
    P.meta = dict(grid=(gx, gy, gz), h=h, nb=nb, bs=bs, sigma=sigma, phis=phis, vox=vox, n_ptv=int(is_ptv.sum()),
                  n_oar1=int(is_o1.sum()), n_oar2=int(is_o2.sum()), c1=c1, c2=c2)
    return P


# ---- config 5: counter-hash random CSR (pure integer arithmetic; reproducible on a device) -------
_M1, _M2 = np.uint64(0xBF58476D1CE4E5B9), np.uint64(0x94D049BB133111EB)
_K1, _K2 = np.uint64(0x9E3779B97F4A7C15), np.uint64(0xD1B54A32D192ED03)


def _mix64(z):
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def hash3(seed, i, t):
    """h(seed, i, t) = mix64(mix64(seed ^ i*K1) + t*K2); all uint64 wrap-around arithmetic."""
    with np.errstate(over="ignore"):
        return _mix64(_mix64(np.uint64(seed) ^ (np.asarray(i, np.uint64) * _K1)) + np.asarray(t, np.uint64) * _K2)


def random_csr(m: int, k: int, seed: int):
    """Row i has k distinct sorted columns, one per stratum: col_t = t*(n/k) + h(seed,i,t) mod (n/k), n = m/2
    (uniform within each stratum, distinct and sorted by construction); value = ((h>>40) + 1) / 2^24 in (0,1]."""
    n = m // 2
    assert n % k == 0, "n must be a multiple of k"
    w = np.uint64(n // k)
    i = np.arange(m, dtype=np.uint64)[:, None]
    t = np.arange(k, dtype=np.uint64)[None, :]
    h = hash3(seed, i, t)
    col = (t * w + h % w).astype(np.int32).ravel()
    val = (((h >> np.uint64(40)) + np.uint64(1)).astype(np.float64) / 2.0**24).astype(np.float32).ravel()
    rowptr = np.arange(m + 1, dtype=np.int64) * k
    return rowptr, col, val


def config5_sweep_point(log2m=16, k=16, with_tv=True, n_sweeps=20, N=5, seed=SEED0 + 5) -> Problem:
    """BASELINE.json configs[4]: one point of the hyperslab-projection throughput sweep (consistent by construction)."""
    m = 1 << log2m
    n = m // 2
    rowptr, col, val = random_csr(m, k, seed)
    u = lambda tag, cnt: ((hash3(seed + tag, np.arange(cnt, dtype=np.uint64), 0) >> np.uint64(40)) + np.uint64(1)).astype(np.float64) / 2.0**24
    x_star = u(1, n).astype(np.float32)
    delta = np.maximum(0.1 * u(2, m), 1e-3)  # U(0,0.1) floored at 1e-3 so that x* stays strictly inside in fp32 too
    P = Problem(f"cfg5_m2^{log2m}_k{k}", m, n, rowptr, col, val, None, None, np.zeros(n, np.float32), np.ones(n, np.float32), np.zeros(n, np.float32))
    ax = P.scipy() @ x_star.astype(np.float64)
    # bounds rounded outward with one extra fp32 ulp so that x* stays feasible under any summation order
    P.lb = np.nextafter(_f32_down(ax - delta), np.float32(-np.inf))
    P.ub = np.nextafter(_f32_up(ax + delta), np.float32(np.inf))
    P.x_true = x_star
    P.objective, P.shape = ("tv1d", (n,)) if with_tv else (None, None)
    P.n_sweeps, P.N, P.beta0, P.a, P.lam = n_sweeps, (N if with_tv else 0), 1.0, 0.99, 1.0
    P.meta = dict(k=k, log2m=log2m)
    return P
