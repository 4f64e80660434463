"""Builder's CPU restatement of the superiorized sweep -- REPORTED BASELINES, neither the oracle nor the product.

bench.py times these beside the GPU path (CPU baselines item 2):
  * scipy:  the paper's own CPU structure ("NumPy and SciPy.sparse ... for CPU"): fp32 csr_matrix products
            y = d * viol(A @ x), x = clip(x - lam * (AT @ y)) plus a NumPy isotropic-TV perturbation phase; SciPy's CSR
            mat-vec is single-threaded, so this is ONE core.
  * openmp: the same sweep as plain fp64 loops in C with OpenMP (row-parallel forward product, row-parallel product with an
            explicit transposed CSR), on ALL host cores (baseline/_cpu_csr.c).
Nothing here is imported by the library, the tests' parity checks or the oracle.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


def _tv2d_value_grad(X):
    dx = np.zeros_like(X)
    dy = np.zeros_like(X)
    dx[:-1, :-1] = X[1:, :-1] - X[:-1, :-1]
    dy[:-1, :-1] = X[:-1, 1:] - X[:-1, :-1]
    t = np.sqrt(dx * dx + dy * dy)
    with np.errstate(divide="ignore", invalid="ignore"):
        ux = np.where(t > 0, dx / t, 0.0)
        uy = np.where(t > 0, dy / t, 0.0)
    g = -(ux + uy)
    g[1:, :] += ux[:-1, :]
    g[:, 1:] += uy[:, :-1]
    return float(t.sum()), g


def _tv2d_value(X):
    dx = X[1:, :-1] - X[:-1, :-1]
    dy = X[:-1, 1:] - X[:-1, :-1]
    return float(np.sqrt(dx * dx + dy * dy).sum())


def perturb_tv2d(x, shape, ell, N, beta0, a):
    """Alg. 1 lines 4-17 with the TV objective in NumPy (fp64 values, PER_TRIAL exponent)."""
    X = x.reshape(shape).astype(np.float64)
    fx = _tv2d_value(X)
    for _ in range(N):
        _, g = _tv2d_value_grad(X)
        s = float(np.sqrt((g * g).sum()))
        for _trial in range(10000):
            beta = beta0 * a**ell
            ell += 1
            Z = X - (beta / s) * g if s > 0 else X
            fz = _tv2d_value(Z)
            if fz <= fx:
                X, fx = Z, fz
                break
    return X.ravel().astype(x.dtype), ell


def time_scipy(P, budget_s=10.0):
    """sweeps/s of the SciPy fp32 restatement on the first sweeps of the workload (1 core)."""
    import scipy.sparse as sp

    ip = P.rowptr.astype(np.int32) if P.nnz < 2**31 else P.rowptr
    A = sp.csr_matrix((P.val, P.col, ip), shape=(P.m, P.n))
    AT = A.T.tocsr()
    rho = np.asarray(A.multiply(A).sum(axis=1)).ravel()
    with np.errstate(over="ignore", divide="ignore"):
        d = np.where(rho > 0, (1.0 / P.m) / np.maximum(rho, 1e-300), 0.0).astype(np.float32)
    x = P.x0.astype(np.float32).copy()
    ell, done = 0, 0
    t0 = time.perf_counter()
    while True:
        if P.objective == "tv2d" and P.N > 0:
            x, ell = perturb_tv2d(x, P.shape, ell, P.N, P.beta0, P.a)
        r = A @ x
        c = np.where(r > P.ub, r - P.ub, np.where(r < P.lb, r - P.lb, 0.0)).astype(np.float32)
        x = np.clip(x - np.float32(P.lam) * (AT @ (d * c)), P.lo, P.hi).astype(np.float32)
        done += 1
        el = time.perf_counter() - t0
        if el >= budget_s or done >= P.n_sweeps or el + el / done > 1.5 * budget_s:
            break
    return done / el, done, el


_lib = None


def _omp():
    global _lib
    if _lib is None:
        src, so = os.path.join(_HERE, "_cpu_csr.c"), os.path.join(_HERE, "_cpu_csr.so")
        if not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
            tmp = f"{so}.{os.getpid()}.tmp"
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, src, "-lm"])
            os.replace(tmp, so)
        _lib = ctypes.CDLL(so)
        _lib.cpu_threads.restype = ctypes.c_int
    return _lib


def time_openmp(P, budget_s=10.0):
    """sweeps/s of the plain fp64 OpenMP sweep (all host cores) + the NumPy TV phase, same protocol as time_scipy."""
    import scipy.sparse as sp

    L = _omp()
    ip = P.rowptr.astype(np.int32) if P.nnz < 2**31 else P.rowptr
    AT = sp.csr_matrix((P.val, P.col, ip), shape=(P.m, P.n)).T.tocsr()
    AT.sort_indices()
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    f8 = lambda a: np.ascontiguousarray(a, np.float64)
    rp, col, val = np.ascontiguousarray(P.rowptr, np.int64), np.ascontiguousarray(P.col, np.int32), f8(P.val)
    trp, tcol, tval = np.ascontiguousarray(AT.indptr, np.int64), np.ascontiguousarray(AT.indices, np.int32), f8(AT.data)
    lb, ub, lo, hi = f8(P.lb), f8(P.ub), f8(P.lo), f8(P.hi)
    d, y = np.zeros(P.m), np.zeros(P.m)
    L.cpu_setup(ctypes.c_int64(P.m), p(rp), p(val), p(d))
    x = f8(P.x0).copy()
    ell, done = 0, 0
    t0 = time.perf_counter()
    while True:
        if P.objective == "tv2d" and P.N > 0:
            x, ell = perturb_tv2d(x, P.shape, ell, P.N, P.beta0, P.a)
            x = f8(x)
        L.cpu_sweep(ctypes.c_int64(P.m), ctypes.c_int64(P.n), p(rp), p(col), p(val), p(trp), p(tcol), p(tval), p(lb), p(ub), p(d), p(lo),
                    p(hi), ctypes.c_double(P.lam), p(x), p(y))
        done += 1
        el = time.perf_counter() - t0
        if el >= budget_s or done >= P.n_sweeps or el + el / done > 1.5 * budget_s:
            break
    return done / el, done, el, int(L.cpu_threads())
