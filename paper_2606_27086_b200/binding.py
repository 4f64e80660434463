"""ctypes binding of libsup.so -- same names as include/sup.h, argument marshalling only."""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_double, c_int, c_int8, c_int32, c_int64, c_size_t, c_void_p

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libsup.so")
_lib = None

F32, F64 = 0, 1
OBJ_NONE, OBJ_TV2D, OBJ_TV1D, OBJ_DOSE, OBJ_MEAN, OBJ_TV3D = 0, 1, 2, 3, 4, 5
PER_TRIAL, PER_SWEEP = 0, 1
WS_CREATE, WS_BLOCKS, WS_DOSE = 0, 1, 2
_OBJ = {None: OBJ_NONE, "none": OBJ_NONE, "tv2d": OBJ_TV2D, "tv1d": OBJ_TV1D, "dose": OBJ_DOSE, "mean": OBJ_MEAN, "tv3d": OBJ_TV3D}


class SupError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"libsup status {status}: {msg}")
        self.status = status


class _Csr(Structure):
    _fields_ = [("m", c_int64), ("n", c_int64), ("nnz", c_int64), ("rowptr", c_void_p), ("col", c_void_p), ("val", c_void_p)]


class _Options(Structure):
    _fields_ = [("objective", c_int), ("shape", c_int64 * 3), ("lambda_", c_double), ("block_iterative", c_int),
                ("step_policy", c_int), ("ell0", c_int64), ("k0", c_int64), ("trace_mode", c_int), ("trace", c_void_p),
                ("decisions", c_void_p), ("decision_f", c_void_p), ("decisions_cap", c_int64), ("use_graph", c_int),
                ("n_restart", c_int64), ("algorithm", c_int), ("stop_enabled", c_int), ("prox_tol", c_double),
                ("dprox_tol", c_double), ("n_consec", c_int), ("dobj_tol", c_double), ("step_rule", c_int), ("f_ref", c_double),
                ("f_ref_shrink", c_double)]


class _State(Structure):
    _fields_ = [("ell", c_int64), ("k", c_int64), ("n_trials", c_int64), ("n_decisions", c_int64), ("warn", c_int32),
                ("fault", c_int32), ("f", c_double), ("n_done", c_int64), ("stop_reason", c_int32), ("step", c_double), ("f_ref", c_double)]


def lib():
    """Loads libsup.so (building it in-tree with nvcc if it is missing).  Raises if that is impossible."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            from .build import build_lib

            build_lib()
        L = ctypes.CDLL(_LIBPATH)
        L.sup_version.restype = c_char_p
        L.sup_last_error.restype = c_char_p
        L.sup_last_error.argtypes = [c_void_p]
        L.sup_launch_count.restype = c_int64
        L.sup_launch_count.argtypes = [c_void_p]
        L.sup_workspace_bytes.argtypes = [c_int, c_int64, c_int64, c_int64, c_int, c_int, POINTER(c_size_t), POINTER(c_size_t)]
        L.sup_create.argtypes = [POINTER(c_void_p), POINTER(_Csr), c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int,
                                 c_void_p, c_size_t, c_void_p, c_size_t, c_void_p]
        L.sup_destroy.argtypes = [c_void_p]
        L.sup_set_blocks.argtypes = [c_void_p, c_int, POINTER(c_int64), c_void_p, c_size_t, c_void_p, c_size_t]
        L.sup_set_dose_matrix.argtypes = [c_void_p, POINTER(_Csr), c_void_p, c_size_t, c_void_p, c_size_t]
        L.sup_project_simultaneous.argtypes = [c_void_p, c_void_p, c_double, c_int]
        L.sup_block_iterative.argtypes = [c_void_p, c_void_p, c_double, c_int]
        L.sup_forward_violation.argtypes = [c_void_p, c_void_p]
        L.sup_backproject_update.argtypes = [c_void_p, c_void_p, c_double]
        L.sup_perturb_tv.argtypes = [c_void_p, c_void_p, c_int, POINTER(c_int64), c_int, c_double, c_double, POINTER(c_int64)]
        L.sup_perturb_dose.argtypes = [c_void_p, c_void_p, c_int, c_double, c_double, POINTER(c_int64)]
        L.sup_perturb_mean.argtypes = [c_void_p, c_void_p, c_int, c_double, c_double, POINTER(c_int64)]
        L.sup_set_dose_mode.argtypes = [c_void_p, c_int]
        L.sup_set_perturb_mode.argtypes = [c_void_p, c_int]
        L.sup_tv2d_value_static.argtypes = [c_void_p, c_int, c_int64, c_int64, c_void_p, c_void_p]
        L.sup_perturb_adaptive.argtypes = [c_void_p, c_void_p, c_int, POINTER(c_int64), c_int, POINTER(c_double), c_double]
        L.sup_project_drop.argtypes = [c_void_p, c_void_p, c_double, c_int]
        L.sup_backproject_partial.argtypes = [c_void_p, c_void_p, c_double]
        L.sup_apply_update.argtypes = [c_void_p, c_void_p, c_void_p, c_double]
        L.sup_project_emr.argtypes = [c_void_p, c_void_p, c_int]
        L.sup_superiorize.argtypes = [c_void_p, c_void_p, c_int, c_int, c_double, c_double, POINTER(_Options)]
        L.sup_superiorize_host.argtypes = [c_void_p, c_void_p, c_int, c_int, c_double, c_double, POINTER(_Options)]
        L.sup_get_state.argtypes = [c_void_p, POINTER(_State)]
        L.sup_proximity.argtypes = [c_void_p, c_void_p, c_int, c_double, POINTER(c_double)]
        L.sup_objective.argtypes = [c_void_p, c_void_p, c_int, POINTER(c_int64), POINTER(c_double)]
        L.sup_get_derived.argtypes = [c_void_p, c_int, c_void_p, c_size_t]
        L.sup_set_row_mode.argtypes = [c_void_p, c_int, c_int]
        L.sup_set_layout.argtypes = [c_void_p, POINTER(c_int64), POINTER(c_int64)]
        for f in ("sup_workspace_bytes", "sup_create", "sup_destroy", "sup_set_blocks", "sup_set_dose_matrix",
                  "sup_project_simultaneous", "sup_block_iterative", "sup_forward_violation", "sup_backproject_update", "sup_perturb_tv", "sup_perturb_dose", "sup_superiorize",
                  "sup_superiorize_host", "sup_get_state", "sup_proximity", "sup_objective", "sup_get_derived", "sup_set_row_mode", "sup_set_layout", "sup_perturb_mean", "sup_project_drop", "sup_project_emr", "sup_backproject_partial", "sup_apply_update"):
            getattr(L, f).restype = c_int
        _lib = L
    return _lib


def _dev(a, dtype, device):
    """numpy / torch -> contiguous torch tensor of `dtype` on `device` (no copy when already there)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        a = torch.from_numpy(np.ascontiguousarray(a))
    return a.to(device=device, dtype=dtype).contiguous()


def _ptr(t):
    return None if t is None else c_void_p(t.data_ptr())


def _bytes_tensor(nbytes, device):
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def sup_workspace_bytes(kind, m, n, nnz, dtype=F32, n_blocks=1):
    p, s = c_size_t(0), c_size_t(0)
    rc = lib().sup_workspace_bytes(kind, m, n, nnz, dtype, n_blocks, byref(p), byref(s))
    if rc:
        raise SupError(rc, lib().sup_last_error(None).decode())
    return p.value, s.value


class SupHandle:
    """Owns the device tensors a sup_handle borrows (matrix, bounds, workspace) and the stream it runs on."""

    def __init__(self):
        self.h = c_void_p(None)
        self.keep = []
        self.stream = None
        self.device = None
        self.tdtype = torch.float32
        self.dtype = F32
        self.m = self.n = self.nnz = 0

    def _check(self, rc):
        if rc:
            raise SupError(rc, lib().sup_last_error(self.h).decode())

    def _enter(self):
        self.stream.wait_stream(torch.cuda.current_stream(self.device))

    def _exit(self):
        torch.cuda.current_stream(self.device).wait_stream(self.stream)

    def x_tensor(self, x):
        return _dev(x, self.tdtype, self.device).clone() if not (isinstance(x, torch.Tensor) and x.is_cuda) else x

    @property
    def launches(self):
        return int(lib().sup_launch_count(self.h))

    def __del__(self):
        try:
            sup_destroy(self)
        except Exception:
            pass


def _csr(rowptr, col, val, n, tdtype, device):
    rp = _dev(rowptr, torch.int64, device)
    c = _dev(col, torch.int32, device)
    v = _dev(val, tdtype, device)
    m = rp.numel() - 1
    s = _Csr(m, n, v.numel(), rp.data_ptr(), c.data_ptr(), v.data_ptr())
    return s, (rp, c, v)


def sup_create(rowptr, col, val, lb, ub, box_lo, box_hi, weights=None, dtype=F32, n=None, device="cuda:0") -> SupHandle:
    """sup_create(A_csr, lb, ub, box, weights): arrays may be numpy or torch; they are moved to `device` once."""
    if not torch.cuda.is_available():
        raise SupError(4, "no CUDA device: libsup has no CPU fallback")
    H = SupHandle()
    H.device = torch.device(device)
    H.dtype = dtype
    H.tdtype = torch.float32 if dtype == F32 else torch.float64
    with torch.cuda.device(H.device):
        H.stream = torch.cuda.Stream(device=H.device)
        lo = _dev(box_lo, H.tdtype, H.device)
        n = int(lo.numel()) if n is None else int(n)
        A, keepA = _csr(rowptr, col, val, n, H.tdtype, H.device)
        lb_t, ub_t, hi = _dev(lb, H.tdtype, H.device), _dev(ub, H.tdtype, H.device), _dev(box_hi, H.tdtype, H.device)
        w = _dev(weights, H.tdtype, H.device)
        H.m, H.n, H.nnz = int(A.m), n, int(A.nnz)
        pb, sb = sup_workspace_bytes(WS_CREATE, H.m, H.n, H.nnz, dtype)
        ws, scratch = _bytes_tensor(pb, H.device), _bytes_tensor(sb, H.device)
        H.keep += [keepA, lb_t, ub_t, lo, hi, w, ws]
        H._enter()
        rc = lib().sup_create(byref(H.h), byref(A), _ptr(lb_t), _ptr(ub_t), _ptr(lo), _ptr(hi), _ptr(w), dtype, _ptr(ws),
                              ws.numel(), _ptr(scratch), scratch.numel(), c_void_p(H.stream.cuda_stream))
        if rc:
            raise SupError(rc, lib().sup_last_error(None).decode())
        H._exit()
        del scratch
    return H


def sup_destroy(H: SupHandle):
    if H.h:
        lib().sup_destroy(H.h)
        H.h = c_void_p(None)
        H.keep = []


def sup_set_blocks(H: SupHandle, block_rowptr):
    br = np.ascontiguousarray(block_rowptr, np.int64)
    nb = br.size - 1
    pb, sb = sup_workspace_bytes(WS_BLOCKS, H.m, H.n, H.nnz, H.dtype, nb)
    ws, scratch = _bytes_tensor(pb, H.device), _bytes_tensor(sb, H.device)
    H.keep.append(ws)
    H._enter()
    H._check(lib().sup_set_blocks(H.h, nb, br.ctypes.data_as(POINTER(c_int64)), _ptr(ws), ws.numel(), _ptr(scratch), scratch.numel()))
    H._exit()


def sup_set_dose_matrix(H: SupHandle, rowptr, col, val):
    D, keepD = _csr(rowptr, col, val, H.n, H.tdtype, H.device)
    pb, sb = sup_workspace_bytes(WS_DOSE, int(D.m), H.n, int(D.nnz), H.dtype)
    ws, scratch = _bytes_tensor(pb, H.device), _bytes_tensor(sb, H.device)
    H.keep += [keepD, ws]
    H._enter()
    H._check(lib().sup_set_dose_matrix(H.h, byref(D), _ptr(ws), ws.numel(), _ptr(scratch), scratch.numel()))
    H._exit()


def sup_set_layout(H: SupHandle, x_shape=None, y_shape=None):
    """x_shape = (rows, cols) of the image x is, y_shape = (angles, bins) of the sinogram the rows of A are; None = no hint."""
    arr = lambda s: None if s is None else (c_int64 * 2)(int(s[0]), int(s[1]))
    H._enter()
    H._check(lib().sup_set_layout(H.h, arr(x_shape), arr(y_shape)))
    H._exit()


def sup_set_row_mode(H: SupHandle, lanes_forward=-1, lanes_backward=-1):
    H._enter()
    H._check(lib().sup_set_row_mode(H.h, int(lanes_forward), int(lanes_backward)))
    H._exit()


def sup_project_simultaneous(H: SupHandle, x: torch.Tensor, lam=1.0, n_sweeps=1):
    H._enter()
    H._check(lib().sup_project_simultaneous(H.h, _ptr(x), lam, n_sweeps))
    H._exit()
    return x


def sup_forward_violation(H: SupHandle, x: torch.Tensor, sync_streams=True):
    if sync_streams:
        H._enter()
    H._check(lib().sup_forward_violation(H.h, _ptr(x)))
    if sync_streams:
        H._exit()


def sup_backproject_update(H: SupHandle, x: torch.Tensor, lam=1.0, sync_streams=True):
    if sync_streams:
        H._enter()
    H._check(lib().sup_backproject_update(H.h, _ptr(x), lam))
    if sync_streams:
        H._exit()


def sup_backproject_partial(H: SupHandle, u: torch.Tensor, scale=1.0):
    H._enter()
    H._check(lib().sup_backproject_partial(H.h, _ptr(u), scale))
    H._exit()
    return u


def sup_apply_update(H: SupHandle, x: torch.Tensor, u: torch.Tensor, lam=1.0):
    H._enter()
    H._check(lib().sup_apply_update(H.h, _ptr(x), _ptr(u), lam))
    H._exit()
    return x


def sup_project_drop(H: SupHandle, x: torch.Tensor, lam=1.0, n_sweeps=1):
    H._enter()
    H._check(lib().sup_project_drop(H.h, _ptr(x), lam, n_sweeps))
    H._exit()
    return x


def sup_project_emr(H: SupHandle, x: torch.Tensor, n_sweeps=1):
    H._enter()
    H._check(lib().sup_project_emr(H.h, _ptr(x), n_sweeps))
    H._exit()
    return x


def sup_block_iterative(H: SupHandle, x: torch.Tensor, lam=1.0, n_sweeps=1):
    H._enter()
    H._check(lib().sup_block_iterative(H.h, _ptr(x), lam, n_sweeps))
    H._exit()
    return x


def sup_perturb_tv(H: SupHandle, x: torch.Tensor, shape, N, beta0, a, ell=0):
    shape = tuple(int(s) for s in shape)
    sh = (c_int64 * 3)(*(list(shape) + [0] * (3 - len(shape))))
    e = c_int64(int(ell))
    H._enter()
    H._check(lib().sup_perturb_tv(H.h, _ptr(x), len(shape), sh, N, beta0, a, byref(e)))
    H._exit()
    return e.value


def sup_perturb_dose(H: SupHandle, x: torch.Tensor, N, beta0, a, ell=0):
    e = c_int64(int(ell))
    H._enter()
    H._check(lib().sup_perturb_dose(H.h, _ptr(x), N, beta0, a, byref(e)))
    H._exit()
    return e.value


ALG_DEFAULT, ALG_DROP, ALG_EMR = 0, 2, 3
_ALG = {None: ALG_DEFAULT, "sim": ALG_DEFAULT, "block": ALG_DEFAULT, "drop": ALG_DROP, "emr": ALG_EMR}


def sup_perturb_mean(H: SupHandle, x: torch.Tensor, N, beta0, a, ell=0):
    e = c_int64(int(ell))
    H._enter()
    H._check(lib().sup_perturb_mean(H.h, _ptr(x), N, beta0, a, byref(e)))
    H._exit()
    return e.value


def sup_set_perturb_mode(H: SupHandle, mode: int):
    """0: small TV2D images take the cluster kernel (default); 1: always the cooperative grid kernel."""
    H._check(lib().sup_set_perturb_mode(H.h, int(mode)))


def sup_set_dose_mode(H: SupHandle, mode: int):
    """0: the dose perturbation through the Gram matrix when it was built (default); 1: by matrix passes over D and D^T."""
    H._check(lib().sup_set_dose_mode(H.h, int(mode)))


def sup_perturb_adaptive(H: SupHandle, x: torch.Tensor, objective, N, f_ref, shrink=0.5, shape=None):
    """One phase with Eq. 11's step size; returns the updated reference value."""
    k = _OBJ[objective] if not isinstance(objective, int) else objective
    sh = (c_int64 * 3)(*(list(shape) + [0] * (3 - len(shape)))) if shape is not None else None
    fr = c_double(float(f_ref))
    H._enter()
    H._check(lib().sup_perturb_adaptive(H.h, _ptr(x), k, sh, int(N), byref(fr), c_double(float(shrink))))
    H._exit()
    return fr.value


def _options(H, objective, shape, lam, block, policy, ell0, k0, trace, decisions, decision_f, use_graph, n_restart=0, algorithm=None,
             stop=None, adaptive=None):
    o = _Options()
    o.objective = _OBJ[objective] if not isinstance(objective, int) else objective
    if shape is not None and o.objective == OBJ_TV2D:
        o.shape[0], o.shape[1] = int(shape[0]), int(shape[1])
    if shape is not None and o.objective == OBJ_TV3D:
        o.shape[0], o.shape[1], o.shape[2] = int(shape[0]), int(shape[1]), int(shape[2])
    o.lambda_ = lam
    o.block_iterative = int(bool(block))
    o.step_policy = policy
    o.ell0, o.k0 = int(ell0), int(k0)
    o.trace_mode = int(trace is not None)
    o.trace = trace.data_ptr() if trace is not None else None
    o.decisions = decisions.data_ptr() if decisions is not None else None
    o.decision_f = decision_f.data_ptr() if decision_f is not None else None
    o.decisions_cap = int(decisions.numel()) if decisions is not None else (int(decision_f.shape[0]) if decision_f is not None else 0)
    o.use_graph = int(bool(use_graph))
    o.n_restart = int(n_restart)
    o.algorithm = _ALG[algorithm] if not isinstance(algorithm, int) else algorithm
    if stop is not None:  # dict(prox_tol, dprox_tol, n_consec, dobj_tol): the paper's defaults where a key is missing
        o.stop_enabled = 1
        o.prox_tol, o.dprox_tol = float(stop.get("prox_tol", 1e-6)), float(stop.get("dprox_tol", 1e-8))
        o.n_consec, o.dobj_tol = int(stop.get("n_consec", 5)), float(stop.get("dobj_tol", 1e-6))
    if adaptive is not None:  # dict(f_ref, shrink): Eq. 11's step size (SUP_RULE_ADAPTIVE)
        o.step_rule, o.f_ref, o.f_ref_shrink = 1, float(adaptive["f_ref"]), float(adaptive.get("shrink", 0.5))
    return o


def sup_superiorize(H: SupHandle, x: torch.Tensor, n_iter, N, beta0, a, objective=None, shape=None, lam=1.0, block=False,
                    policy=PER_TRIAL, ell0=0, k0=0, trace=None, decisions=None, decision_f=None, use_graph=True, n_restart=0,
                    algorithm=None, stop=None, adaptive=None):
    """Algorithm 1 on device tensor x (in place, asynchronous).  trace: float64 [n_iter,4] device tensor or None;
    decisions: int8 [cap] device tensor or None; decision_f: float64 [cap,2] device tensor or None."""
    o = _options(H, objective, shape, lam, block, policy, ell0, k0, trace, decisions, decision_f, use_graph, n_restart, algorithm, stop, adaptive)
    H._enter()
    H._check(lib().sup_superiorize(H.h, _ptr(x), n_iter, N, beta0, a, byref(o)))
    H._exit()
    return x


def sup_superiorize_host(H: SupHandle, x_host: torch.Tensor, n_iter, N, beta0, a, objective=None, shape=None, lam=1.0,
                         block=False, policy=PER_TRIAL, ell0=0, k0=0, use_graph=True, n_restart=0):
    """Same with x a (pinned) HOST tensor: H2D copy, run, D2H copy, synchronise -- the end-to-end entry."""
    assert not x_host.is_cuda and x_host.dtype == H.tdtype and x_host.is_contiguous()
    o = _options(H, objective, shape, lam, block, policy, ell0, k0, None, None, None, use_graph, n_restart)
    H._enter()
    H._check(lib().sup_superiorize_host(H.h, c_void_p(x_host.data_ptr()), n_iter, N, beta0, a, byref(o)))
    H._exit()
    return x_host


def sup_get_state(H: SupHandle) -> dict:
    s = _State()
    H._check(lib().sup_get_state(H.h, byref(s)))
    return dict(ell=s.ell, k=s.k, n_trials=s.n_trials, n_decisions=s.n_decisions, warn=s.warn, fault=s.fault, f=s.f,
                n_done=s.n_done, stop_reason=s.stop_reason, step=s.step, f_ref=s.f_ref)


def sup_proximity(H: SupHandle, x: torch.Tensor, mode=0, p=2.0) -> float:
    out = c_double(0.0)
    H._enter()
    H._check(lib().sup_proximity(H.h, _ptr(x), mode, p, byref(out)))
    H._exit()
    return out.value


def sup_objective(H: SupHandle, x: torch.Tensor, kind, shape=None) -> float:
    k = _OBJ[kind] if not isinstance(kind, int) else kind
    sh = (c_int64 * 3)(*(list(shape) + [0] * (3 - len(shape)))) if shape is not None else None
    out = c_double(0.0)
    H._enter()
    H._check(lib().sup_objective(H.h, _ptr(x), k, sh, byref(out)))
    H._exit()
    return out.value


STATIC_MAX_ROWS = 16384


def sup_tv2d_value_static(x: torch.Tensor, shape, out: torch.Tensor = None, sync=True):
    """TV2D value of the device tensor x (float32 / float64, ny*nx elements) through the entry point that allocates nothing
    (sup_tv2d_value_static; scratch in a static device array, at most STATIC_MAX_ROWS rows).  out: a device float64 tensor of one
    element (allocated here when None -- the C entry itself takes it from the caller).  Runs on torch's current stream.
    Returns the value as a float when sync, else `out`."""
    assert x.is_cuda and x.is_contiguous() and x.dtype in (torch.float32, torch.float64)
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=x.device)
    with torch.cuda.device(x.device):
        st = torch.cuda.current_stream(x.device)
        rc = lib().sup_tv2d_value_static(_ptr(x), F32 if x.dtype == torch.float32 else F64, int(shape[0]), int(shape[1]), _ptr(out),
                                         c_void_p(st.cuda_stream))
    if rc:
        raise SupError(rc, lib().sup_last_error(None).decode())
    return float(out.item()) if sync else out


def sup_get_derived(H: SupHandle, which: int) -> torch.Tensor:
    shapes = {0: (H.m, H.tdtype), 1: (H.n + 1, torch.int64), 2: (H.nnz, torch.int32), 3: (H.nnz, H.tdtype), 5: (H.m, H.tdtype)}
    cnt, dt = shapes[which]
    out = torch.empty(cnt, dtype=dt, device=H.device)
    H._enter()
    H._check(lib().sup_get_derived(H.h, which, _ptr(out), out.numel() * out.element_size()))
    H._exit()
    return out


def create_from_problem(P, dtype=F32, device="cuda:0", blocks=True, layout=True) -> SupHandle:
    """Convenience for tests/bench: a gen.Problem -> handle (with blocks / dose matrix when the problem has them).
    layout: pass the problem's geometry (image shape; angles x bins of a CT sinogram) to sup_set_layout."""
    H = sup_create(P.rowptr, P.col, P.val, P.lb, P.ub, P.lo, P.hi, P.weights, dtype=dtype, n=P.n, device=device)
    if layout:
        xs = tuple(P.shape) if P.shape is not None and len(P.shape) == 2 and P.shape[0] * P.shape[1] == P.n else None
        ys = (P.meta["n_angles"], P.meta["n_bins"]) if "n_angles" in P.meta and P.meta["n_angles"] * P.meta["n_bins"] == P.m else None
        if xs is not None or ys is not None:
            sup_set_layout(H, xs, ys)
    if blocks and P.block_rowptr is not None:
        sup_set_blocks(H, P.block_rowptr)
    if P.dose is not None:
        sup_set_dose_matrix(H, P.dose[0], P.dose[1], P.dose[2])
    return H
