"""Row-sharded sweeps over several GPUs: one process per GPU, contiguous row blocks of A
balanced by nonzeros, a replica of x on every GPU, ONE all-reduce of an n-vector per sweep (torch.distributed / NCCL over NVLink).

This module only partitions, marshals and calls the collective; every product, the update and the perturbation run in libsup's
kernels (sup_forward_violation, sup_backproject_partial, sup_apply_update, sup_perturb_tv).  The perturbation phase is replicated:
every rank runs the same deterministic kernel on the same x.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B


def partition_rows(rowptr, world: int):
    """Contiguous row blocks [r_g, r_{g+1}) with (almost) equal numbers of stored entries; returns int64 [world + 1]."""
    rowptr = np.asarray(rowptr, np.int64)
    m, nnz = rowptr.size - 1, int(rowptr[-1])
    cuts = [0]
    for g in range(1, world):
        cuts.append(int(np.searchsorted(rowptr, (nnz * g) // world, side="left")))
    cuts.append(m)
    cuts = np.maximum.accumulate(np.minimum(np.asarray(cuts, np.int64), m))
    return cuts


def row_block(P, r0: int, r1: int):
    """The arrays of rows [r0, r1) of a gen.Problem-like object: (rowptr, col, val, lb, ub)."""
    e0, e1 = int(P.rowptr[r0]), int(P.rowptr[r1])
    return (P.rowptr[r0:r1 + 1] - e0, P.col[e0:e1], P.val[e0:e1], P.lb[r0:r1], P.ub[r0:r1])


class ShardedSup:
    """This rank's block of a row-sharded problem.  `group` is a torch.distributed process group (None: single process, the
    all-reduce is skipped -- used by the single-GPU emulation in the tests, which adds the blocks' shares itself)."""

    def __init__(self, P, rank: int, world: int, dtype=B.F32, device="cuda:0", group=None, y_layout_rows=None):
        self.rank, self.world, self.group = rank, world, group
        self.cuts = partition_rows(P.rowptr, world)
        r0, r1 = int(self.cuts[rank]), int(self.cuts[rank + 1])
        rp, col, val, lb, ub = row_block(P, r0, r1)
        w_all = np.full(P.m, 1.0 / P.m) if P.weights is None else np.asarray(P.weights, np.float64) / float(np.sum(P.weights))
        self.share = float(w_all[r0:r1].sum())  # the block's share of the global weights (a handle normalises over its own rows)
        self.H = B.sup_create(rp, col, val, lb, ub, P.lo, P.hi, None if P.weights is None else P.weights[r0:r1], dtype=dtype, n=P.n,
                              device=device)
        xs = tuple(P.shape) if P.shape is not None and len(P.shape) == 2 and P.shape[0] * P.shape[1] == P.n else None
        ys = None
        if "n_bins" in P.meta and (r1 - r0) % P.meta["n_bins"] == 0 and r1 > r0:  # whole angles: the block is a sinogram too
            ys = ((r1 - r0) // P.meta["n_bins"], P.meta["n_bins"])
        if xs is not None or ys is not None:
            B.sup_set_layout(self.H, xs, ys)
        self.u = torch.zeros(P.n, dtype=self.H.tdtype, device=device)
        self.P = P

    def partial(self, x):
        """y = D c(x) on this block, then this block's share of A^T y into self.u"""
        B.sup_forward_violation(self.H, x)
        B.sup_backproject_partial(self.H, self.u, self.share)
        return self.u

    def sweep(self, x, lam=1.0):
        u = self.partial(x)
        if self.group is not None and self.world > 1:
            torch.distributed.all_reduce(u, op=torch.distributed.ReduceOp.SUM, group=self.group)
        B.sup_apply_update(self.H, x, u, lam)
        return x

    def superiorize(self, x, n_iter, N, beta0, a, lam=1.0, ell=0):
        """Algorithm 1 with the sharded sweep; the TV perturbation phase is replicated on every rank."""
        P = self.P
        for _ in range(n_iter):
            if N > 0 and P.objective in ("tv2d", "tv1d", "tv3d"):
                ell = B.sup_perturb_tv(self.H, x, P.shape if P.objective != "tv1d" else (P.n,), N, beta0, a, ell)
            self.sweep(x, lam)
        return x, ell
