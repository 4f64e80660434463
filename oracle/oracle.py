"""ctypes wrapper of oracle/sup_oracle.c -- the fp64 CPU ORACLE (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package.  Inputs are the fp32-rounded arrays of a gen.Problem, widened exactly
to fp64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sup_oracle.c")
_LIB = os.path.join(_HERE, "_sup_oracle.so")
_lib = None

OBJ_KIND = {None: 0, "none": 0, "tv2d": 1, "tv1d": 2, "dose": 3, "mean": 4, "tv3d": 5}
ALGORITHM = {"sim": 0, "block": 1, "drop": 2, "emr": 3}
PER_TRIAL, PER_SWEEP = 0, 1


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (no -ffast-math, no FMA contraction, no OpenMP: single-threaded scalar code;
    reductions use binary128 accumulators from libgcc's soft-float, see sup_oracle.c)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = f"{_LIB}.{os.getpid()}.tmp"  # build aside and rename: a process that has the old library mapped keeps it
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _L():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_proximity.restype = ctypes.c_double
        _lib.orc_tv2d.restype = ctypes.c_double
        _lib.orc_tv1d.restype = ctypes.c_double
        _lib.orc_dose.restype = ctypes.c_double
        _lib.orc_mean.restype = ctypes.c_double
        _lib.orc_tv3d.restype = ctypes.c_double
        _lib.orc_perturb_phase3.restype = ctypes.c_int64
        _lib.orc_perturb_adaptive_phase.restype = ctypes.c_int64
        _lib.orc_superiorize_ex.restype = ctypes.c_int
        _lib.orc_perturb_phase.restype = ctypes.c_int64
        _lib.orc_setup.restype = ctypes.c_int
        _lib.orc_superiorize.restype = ctypes.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


_i64, _dbl, _int = ctypes.c_int64, ctypes.c_double, ctypes.c_int


class _RunOpt(ctypes.Structure):  # run_opt_t of sup_oracle.c
    _fields_ = [("algorithm", _int), ("stop_enabled", _int), ("prox_tol", _dbl), ("dprox_tol", _dbl), ("n_consec", _int),
                ("dobj_tol", _dbl), ("n_restart", _i64), ("nz", _i64), ("step_rule", _int), ("f_ref", _dbl), ("f_ref_shrink", _dbl)]


class Oracle:
    """fp64 oracle bound to one problem (CSR + bounds + box [+ weights, blocks, dose matrix])."""

    def __init__(self, m, n, rowptr, col, val, lb, ub, lo, hi, weights=None, block_rowptr=None, dose=None,
                 objective=None, shape=None):
        f8 = lambda a: None if a is None else np.ascontiguousarray(a, np.float64)
        self.m, self.n = int(m), int(n)
        self.rowptr = np.ascontiguousarray(rowptr, np.int64)
        self.col = np.ascontiguousarray(col, np.int32)
        self.val = f8(val)
        self.lb, self.ub, self.lo, self.hi = f8(lb), f8(ub), f8(lo), f8(hi)
        self.w = np.empty(self.m)
        self.rho = np.empty(self.m)
        self.d = np.empty(self.m)
        rc = _L().orc_setup(_i64(self.m), _p(self.rowptr), _p(self.col), _p(self.val), _p(f8(weights)), _p(self.w),
                            _p(self.rho), _p(self.d))
        if rc:
            raise ValueError("weights must be > 0")
        self.block_rowptr = None if block_rowptr is None else np.ascontiguousarray(block_rowptr, np.int64)
        self.objective = objective
        self.shape = shape
        if dose is not None:
            self.d_rowptr = np.ascontiguousarray(dose[0], np.int64)
            self.d_col = np.ascontiguousarray(dose[1], np.int32)
            self.d_val = f8(dose[2])
            self.md = int(dose[3])
        else:
            self.d_rowptr = self.d_col = self.d_val = None
            self.md = 0

    @classmethod
    def from_problem(cls, P, blocks=True):
        return cls(P.m, P.n, P.rowptr, P.col, P.val, P.lb, P.ub, P.lo, P.hi, P.weights,
                   P.block_rowptr if blocks else None, P.dose, P.objective, P.shape)

    # ---- feasibility-seeking --------------------------------------------------------------
    def sweep(self, x, lam=1.0, n_sweeps=1):
        x = np.array(x, np.float64)
        for _ in range(n_sweeps):
            _L().orc_sweep(_i64(self.m), _i64(self.n), _p(self.rowptr), _p(self.col), _p(self.val), _p(self.lb),
                           _p(self.ub), _p(self.d), _p(self.lo), _p(self.hi), _dbl(lam), _p(x))
        return x

    def block_sweep(self, x, lam=1.0, n_sweeps=1, block_rowptr=None):
        br = self.block_rowptr if block_rowptr is None else np.ascontiguousarray(block_rowptr, np.int64)
        x = np.array(x, np.float64)
        for _ in range(n_sweeps):
            _L().orc_block_sweep(_i64(self.m), _i64(self.n), _p(self.rowptr), _p(self.col), _p(self.val), _p(self.lb),
                                 _p(self.ub), _p(self.w), _p(self.d), _p(self.lo), _p(self.hi), _dbl(lam),
                                 _int(br.size - 1), _p(br), _p(x))
        return x

    def drop_sweep(self, x, lam=1.0, n_sweeps=1):
        """DROP, Table A.5: x - lam Z A^T M c(x), then the box."""
        x = np.array(x, np.float64)
        for _ in range(n_sweeps):
            _L().orc_drop_sweep(_i64(self.m), _i64(self.n), _p(self.rowptr), _p(self.col), _p(self.val), _p(self.lb),
                                _p(self.ub), _p(self.w), _p(self.lo), _p(self.hi), _dbl(lam), _p(x))
        return x

    def emr_sweep(self, x, n_sweeps=1, return_step=False):
        """EMR, Table A.5: x - (||p||^2 / ||M^(1/2) A p||^2) p, p = A^T M c(x), then the box."""
        x = np.array(x, np.float64)
        step = _dbl(0.0)
        for _ in range(n_sweeps):
            _L().orc_emr_sweep(_i64(self.m), _i64(self.n), _p(self.rowptr), _p(self.col), _p(self.val), _p(self.lb),
                               _p(self.ub), _p(self.w), _p(self.lo), _p(self.hi), _p(x), ctypes.byref(step))
        return (x, step.value) if return_step else x

    def proximity(self, x, mode=0, p=2.0):
        x = np.ascontiguousarray(x, np.float64)
        return _L().orc_proximity(_i64(self.m), _p(self.rowptr), _p(self.col), _p(self.val), _p(self.lb), _p(self.ub),
                                  _p(self.w), _p(self.rho), _p(x), _int(mode), _dbl(p))

    # ---- objectives -----------------------------------------------------------------------
    def _obj_args(self, kind=None, shape=None):
        kind = self.objective if kind is None else kind
        shape = self.shape if shape is None else shape
        k = OBJ_KIND[kind]
        ny, nx = (shape if k == 1 else (tuple(shape)[1:] if k == 5 else (0, 0)))
        return (_int(k), _i64(ny), _i64(nx), _i64(self.md), _p(self.d_rowptr), _p(self.d_col), _p(self.d_val))

    def objective_value(self, x, kind=None, shape=None):
        kind = self.objective if kind is None else kind
        shape = self.shape if shape is None else shape
        x = np.ascontiguousarray(x, np.float64)
        L = _L()
        if kind == "tv2d":
            return L.orc_tv2d(_p(x), _i64(shape[0]), _i64(shape[1]))
        if kind == "tv1d":
            return L.orc_tv1d(_p(x), _i64(x.size))
        if kind == "dose":
            return L.orc_dose(_i64(self.md), _p(self.d_rowptr), _p(self.d_col), _p(self.d_val), _p(x))
        if kind == "mean":
            return L.orc_mean(_i64(self.md), _p(self.d_rowptr), _p(self.d_col), _p(self.d_val), _p(x))
        if kind == "tv3d":
            return L.orc_tv3d(_p(x), _i64(shape[0]), _i64(shape[1]), _i64(shape[2]))
        return 0.0

    def objective_grad(self, x, kind=None, shape=None):
        kind = self.objective if kind is None else kind
        shape = self.shape if shape is None else shape
        x = np.ascontiguousarray(x, np.float64)
        g = np.zeros_like(x)
        L = _L()
        if kind == "tv2d":
            L.orc_tv2d_grad(_p(x), _i64(shape[0]), _i64(shape[1]), _p(g))
        elif kind == "tv1d":
            L.orc_tv1d_grad(_p(x), _i64(x.size), _p(g))
        elif kind == "dose":
            L.orc_dose_grad(_i64(self.md), _i64(self.n), _p(self.d_rowptr), _p(self.d_col), _p(self.d_val), _p(x), _p(g))
        elif kind == "mean":
            L.orc_mean_grad(_i64(self.md), _i64(self.n), _p(self.d_rowptr), _p(self.d_col), _p(self.d_val), _p(g))
        elif kind == "tv3d":
            L.orc_tv3d_grad(_p(x), _i64(shape[0]), _i64(shape[1]), _i64(shape[2]), _p(g))
        return g

    # ---- perturbation phase / superiorization ---------------------------------------------
    def perturb(self, x, ell, N, beta0, a, k=0, policy=PER_TRIAL, kind=None, shape=None, forced=None, cap=1 << 20):
        """One perturbation phase (Alg. 1 lines 4-17).  Returns dict(x, ell, trials, decisions, margins, fx, warn)."""
        x = np.array(x, np.float64)
        ell_c = _i64(int(ell))
        dec = np.zeros(cap, np.int8)
        mar = np.zeros(cap)
        ndec = _i64(0)
        warn = _int(0)
        fx = _dbl(0.0)
        forced_a = None if forced is None else np.ascontiguousarray(forced, np.int8)
        if (self.objective if kind is None else kind) == "tv3d":
            sh = self.shape if shape is None else shape
            t = _L().orc_perturb_phase3(_i64(self.n), _int(5), _i64(sh[0]), _i64(sh[1]), _i64(sh[2]), _p(x), ctypes.byref(ell_c),
                                        _i64(k), _int(N), _dbl(beta0), _dbl(a), _int(policy), _p(dec), _p(mar), _i64(cap),
                                        ctypes.byref(ndec), _p(forced_a), ctypes.byref(warn), ctypes.byref(fx))
        else:
            t = _L().orc_perturb_phase(_i64(self.n), *self._obj_args(kind, shape), _p(x), ctypes.byref(ell_c), _i64(k),
                                       _int(N), _dbl(beta0), _dbl(a), _int(policy), _p(dec), _p(mar), _i64(cap),
                                       ctypes.byref(ndec), _p(forced_a), ctypes.byref(warn), ctypes.byref(fx))
        nd = min(ndec.value, cap)
        return dict(x=x, ell=ell_c.value, trials=int(t), decisions=dec[:nd].copy(), margins=mar[:nd].copy(), fx=fx.value,
                    warn=warn.value)

    def perturb_adaptive(self, x, N, f_ref, shrink=0.5, kind=None, shape=None, cap=1 << 16):
        """One perturbation phase with Eq. 11's step size (reading A-30).
        Returns dict(x, f_ref (updated), steps, decisions, fx)."""
        kind = self.objective if kind is None else kind
        shape = self.shape if shape is None else shape
        x = np.array(x, np.float64)
        dec = np.zeros(cap, np.int8)
        ndec = _i64(0)
        fr = _dbl(float(f_ref))
        fx = _dbl(0.0)
        oa = self._obj_args(kind, shape)
        nz = int(shape[0]) if kind == "tv3d" else 0
        t = _L().orc_perturb_adaptive_phase(_i64(self.n), _int(OBJ_KIND[kind]), _i64(nz), *oa[1:], _p(x), _int(N), ctypes.byref(fr),
                                            _dbl(shrink), _p(dec), _i64(cap), ctypes.byref(ndec), ctypes.byref(fx))
        return dict(x=x, f_ref=fr.value, steps=int(t), decisions=dec[: min(ndec.value, cap)].copy(), fx=fx.value)

    def superiorize(self, x0, n_iter, N, beta0, a, lam=1.0, policy=PER_TRIAL, block=False, snapshots=(), ell0=0,
                    forced=None, kind=None, shape=None, cap=1 << 22, k0=0, n_restart=0):
        """Algorithm 1 for n_iter sweeps (absolute sweep indices k0 .. k0+n_iter-1; k0 only matters to PER_SWEEP).
        snapshots: sweep counts (1-based: 'after s sweeps') at which x is copied.
        n_restart > 0: restarted perturbations, l <- r at the start of sweep r * n_restart (A-24).
        Returns dict(x, ell, trace[n_iter,4] = (prox0, f, trials, ell), snaps{count: x}, decisions, margins, warn)."""
        x = np.array(x0, np.float64)
        ell = _i64(int(ell0))
        trace = np.zeros((n_iter, 4))
        dec = np.zeros(cap, np.int8)
        mar = np.zeros(cap)
        ndec = _i64(0)
        forced_a = None if forced is None else np.ascontiguousarray(forced, np.int8)
        nb = 0 if not block else self.block_rowptr.size - 1
        snaps = {}
        stops = sorted(set(int(s) for s in snapshots if 0 < int(s) < n_iter)) + [n_iter]
        k = 0
        warn = 0
        for stop in stops:
            cnt = stop - k
            if cnt <= 0:
                continue
            tr = np.zeros((cnt, 4))
            warn |= _L().orc_superiorize(
                _i64(self.m), _i64(self.n), _p(self.rowptr), _p(self.col), _p(self.val), _p(self.lb), _p(self.ub),
                _p(self.w), _p(self.rho), _p(self.d), _p(self.lo), _p(self.hi), _dbl(lam), _int(nb),
                _p(self.block_rowptr) if nb else None, *self._obj_args(kind, shape), _p(x), ctypes.byref(ell), _i64(k0 + k),
                _int(cnt), _int(N), _dbl(beta0), _dbl(a), _int(policy), _p(tr), _p(dec), _p(mar), _i64(cap),
                ctypes.byref(ndec), _p(forced_a), _i64(int(n_restart)))
            trace[k:stop] = tr
            k = stop
            snaps[stop] = x.copy()
        nd = min(ndec.value, cap)
        return dict(x=x, ell=ell.value, trace=trace, snaps=snaps, decisions=dec[:nd].copy(), margins=mar[:nd].copy(),
                    warn=warn)

    def run(self, x0, n_iter, N=0, beta0=1.0, a=0.99, lam=1.0, algorithm="sim", policy=PER_TRIAL, ell0=0, k0=0, kind=None,
            shape=None, n_restart=0, stop=None, forced=None, cap=1 << 22, adaptive=None):
        """Algorithm 1 through orc_superiorize_ex: `algorithm` in {'sim', 'block', 'drop', 'emr'} (Table A.5), any objective
        (incl. 'mean', 'tv3d'), and the paper's stopping rule when stop = dict(prox_tol, dprox_tol, n_consec, dobj_tol)
        (reading A-25).  One call, no snapshots (the rule's counters live inside the call).
        adaptive = dict(f_ref, shrink): Eq. 11's step size instead of the power law (reading A-30); the updated reference
        comes back as 'f_ref'.
        Returns dict(x, ell, n_done, stop_reason, trace[n_done,4], decisions, margins, warn)."""
        kind = self.objective if kind is None else kind
        shape = self.shape if shape is None else shape
        x = np.array(x0, np.float64)
        ell = _i64(int(ell0))
        trace = np.zeros((max(n_iter, 1), 4))
        dec = np.zeros(cap, np.int8)
        mar = np.zeros(cap)
        ndec = _i64(0)
        forced_a = None if forced is None else np.ascontiguousarray(forced, np.int8)
        nb = self.block_rowptr.size - 1 if algorithm == "block" else 0
        opt = _RunOpt(ALGORITHM[algorithm], int(stop is not None), 0.0, 0.0, 0, 0.0, int(n_restart),
                      int(shape[0]) if OBJ_KIND[kind] == 5 else 0)
        if stop is not None:
            opt.prox_tol, opt.dprox_tol = float(stop.get("prox_tol", 1e-6)), float(stop.get("dprox_tol", 1e-8))
            opt.n_consec, opt.dobj_tol = int(stop.get("n_consec", 5)), float(stop.get("dobj_tol", 1e-6))
        if adaptive is not None:
            opt.step_rule, opt.f_ref, opt.f_ref_shrink = 1, float(adaptive["f_ref"]), float(adaptive.get("shrink", 0.5))
        n_done, reason = _int(0), _int(0)
        warn = _L().orc_superiorize_ex(
            _i64(self.m), _i64(self.n), _p(self.rowptr), _p(self.col), _p(self.val), _p(self.lb), _p(self.ub), _p(self.w),
            _p(self.rho), _p(self.d), _p(self.lo), _p(self.hi), _dbl(lam), _int(nb), _p(self.block_rowptr) if nb else None,
            *self._obj_args(kind, shape), _p(x), ctypes.byref(ell), _i64(k0), _int(n_iter), _int(N), _dbl(beta0), _dbl(a),
            _int(policy), _p(trace), _p(dec), _p(mar), _i64(cap), ctypes.byref(ndec), _p(forced_a), ctypes.byref(opt),
            ctypes.byref(n_done), ctypes.byref(reason))
        nd = min(ndec.value, cap)
        return dict(x=x, ell=ell.value, n_done=n_done.value, stop_reason=reason.value, trace=trace[: n_done.value].copy(),
                    decisions=dec[:nd].copy(), margins=mar[:nd].copy(), warn=warn, f_ref=opt.f_ref)
