#!/usr/bin/env python
"""Writes the full-size oracle goldens tests/golden/cfg3_full_*.npz and cfg4_full*.npz.

    python tests/golden/make_goldens.py [cfg3_simul] [cfg3_block] [cfg4] [cfg4_infeasible]     (default: all four)

Imports ONLY gen/ (seeded inputs) and oracle/ (the fp64 CPU oracle): no value below ever comes from the CUDA path.
The oracle needs ~25 s per superiorized sweep at config 3 and ~40 s at config 4 on one core, so the `-m gpu` tests
compare libsup, in the launch configuration bench.py times, against these stored results instead of re-running it.

What is stored per run (PER_TRIAL policy, lambda / N / beta0 / a of the config):
  basic_x<s>          x after s unperturbed sweeps from x0                       (free run; O-SWEEP / O-BLOCK-SWEEP)
  sup_x<s>            x after s superiorized sweeps from x0                      (free run; O-SUPERIORIZE, Alg. 1)
  sup_trace           [S, 4] = proximity (Eq. 5), f(x), #trials, l after each of the S sweeps
  sup_decisions, sup_margins, sup_ell
  step<k>_x           ONE superiorized sweep from the state (fl32(sup_x<k>), l_k, k): what the step-wise parity test of an
                      fp32 handle is compared with (fp64 handles start from sup_x<k> itself and are compared with
                      sup_x<k+1>)
  step<k>_trace, step<k>_decisions, step<k>_margins, step<k>_ell
Arrays that only fp32-mode tests read are stored as fp32 (6e-8 relative, far below the 1e-4 bar) to keep the files small.
"""
from __future__ import annotations

import json
import os
import re
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gen  # noqa: E402
from oracle.oracle import Oracle  # noqa: E402


def fl32(x):
    return np.asarray(x, np.float32).astype(np.float64)


def run(P, block, S, step_ks, f64_keys, tag):
    """free basic run, free superiorized run with snapshots, and one re-synchronised sweep per k in step_ks"""
    O = Oracle.from_problem(P)
    out = {}
    t0 = time.time()
    x = np.array(P.x0, np.float64)
    for s in range(1, S + 1):
        x = O.block_sweep(x, P.lam) if block else O.sweep(x, P.lam)
        if s in (1, S):
            out[f"basic_x{s}"] = x.copy()
        print(f"[{tag}] basic sweep {s}/{S} {time.time() - t0:.0f}s", flush=True)
    snaps = sorted(set([1, S] + [k for k in step_ks if k > 0]))
    R = O.superiorize(P.x0, S, P.N, P.beta0, P.a, lam=P.lam, block=block, snapshots=snaps)
    print(f"[{tag}] superiorized free run {time.time() - t0:.0f}s", flush=True)
    for s in snaps:
        out[f"sup_x{s}"] = R["snaps"][s]
    out["sup_trace"], out["sup_decisions"], out["sup_margins"] = R["trace"], R["decisions"], R["margins"]
    out["sup_ell"] = np.int64(R["ell"])
    for k in step_ks:
        xs = fl32(P.x0 if k == 0 else R["snaps"][k])
        ell = 0 if k == 0 else int(R["trace"][k - 1, 3])
        One = O.superiorize(xs, 1, P.N, P.beta0, P.a, lam=P.lam, block=block, ell0=ell, k0=k)
        out[f"step{k}_x"] = One["x"]
        out[f"step{k}_trace"], out[f"step{k}_decisions"], out[f"step{k}_margins"] = One["trace"], One["decisions"], One["margins"]
        out[f"step{k}_ell"] = np.int64(One["ell"])
        print(f"[{tag}] step from sweep {k} {time.time() - t0:.0f}s", flush=True)
    for key in list(out):  # iterates that only fp32-mode tests read are stored as fp32
        if re.fullmatch(r"(basic_x|sup_x)\d+|step\d+_x", key) and key not in f64_keys:
            out[key] = out[key].astype(np.float32)
    out["meta"] = np.array(json.dumps(dict(
        script="tests/golden/make_goldens.py", problem=P.name, m=P.m, n=P.n, nnz=P.nnz, sweeps=S, N=P.N, beta0=P.beta0, a=P.a,
        lam=P.lam, objective=P.objective, block=bool(block), step_ks=list(step_ks), f64_keys=sorted(f64_keys),
        oracle_seconds=round(time.time() - t0, 1))))
    return out


def main():
    parts = sys.argv[1:] or ["cfg3_simul", "cfg3_block", "cfg4", "cfg4_infeasible"]
    for part in parts:
        if part == "cfg3_simul":
            P = gen.config3_lowdose_ct()
            out = run(P, False, 10, (9,), {"basic_x10", "sup_x1", "sup_x9", "sup_x10"}, part)
            name = "cfg3_full_simul.npz"
        elif part == "cfg3_block":
            P = gen.interleaved_angle_blocks(gen.config3_lowdose_ct(), 16)
            out = run(P, True, 10, (9,), set(), part)
            name = "cfg3_full_block.npz"
        elif part in ("cfg4", "cfg4_infeasible"):
            P = gen.config4_imrt(infeasible=part.endswith("infeasible"))
            out = run(P, False, 5, (4,), {"basic_x1", "basic_x5", "sup_x1", "sup_x4", "sup_x5", "step4_x"}, part)
            name = "cfg4_full" + ("_infeasible" if part.endswith("infeasible") else "") + ".npz"
        else:
            raise SystemExit(f"unknown part {part}")
        np.savez_compressed(os.path.join(HERE, name), **out)
        print(f"wrote {name}: " + ", ".join(f"{k}{getattr(v, 'shape', '')}" for k, v in out.items()), flush=True)


if __name__ == "__main__":
    main()
