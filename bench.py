#!/usr/bin/env python
"""bench.py -- superiorized projection sweeps/s on BASELINE.json's headline workload (512x512 low-dose CT, configs[2]).

    python bench.py --gpus N --steps K --warmup W [--impl ours|reference] [--workload cfg3|cfg1|cfg2|cfg5:<log2m>:<k>]

One "step" = one whole pass of the hot path over the workload: sup_superiorize for the config's sweep count
(cfg3: 100 sweeps, each = perturbation phase of N=5 TV reduction steps + one simultaneous sweep), restarted
from x0.  Prints ONE JSON line (contract in DESIGN.md "Measurement").  N > 1 runs N independent replicas
(the path is single-GPU: "replicas only"), value = all ranks' sweeps / max-over-ranks time; started without a launcher,
`--gpus N` re-executes itself under torch.distributed.run with N ranks and fails if fewer than N devices are visible.

--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
Beside the oracle (cpu_baseline) the line carries two builder's CPU restatements (baseline/cpu_restatement.py): the paper's own
CPU structure in SciPy (1 core) and a plain fp64 OpenMP sweep on all host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "superiorized projection sweeps/s"
UNIT = "sweeps/s"


def load_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def make_problem(name):
    import gen

    if name == "cfg3":
        return gen.config3_lowdose_ct()
    if name.startswith("ct:"):  # ct:<n_pix>:<n_angles>:<n_bins> -- same recipe as cfg3 at another size (experiments)
        _, npx, na, nbn = name.split(":")
        return gen.config3_lowdose_ct(n_pix=int(npx), n_angles=int(na), n_bins=int(nbn))
    if name == "cfg1":
        return gen.config1_tiny_ct()
    if name == "cfg2":
        return gen.config2_crosswell()
    if name == "cfg4":
        return gen.config4_imrt()
    if name.startswith("cfg5"):
        _, lg, k = name.split(":")
        return gen.config5_sweep_point(int(lg), int(k))
    raise SystemExit(f"unknown workload {name}")


WORKLOAD_TEXT = {
    "cfg3": "BASELINE.json configs[2]: low-dose parallel-beam CT 512x512, 720 angles x 729 bins, fp32 CSR + explicit A^T, "
            "TV superiorization N=5 a=0.99, 100 simultaneous sweeps per step",
}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self.stop_flag = False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.samples.append([t.strip() for t in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        sm, mx, reasons = [], 0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            try:
                sm.append(float(s[0]))
                mx = max(mx, float(s[1]))
                for nm, v in zip(names, s[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(sm)}


def dist_setup(world, backend, device=None):
    """One process per GPU (RANK/WORLD_SIZE/MASTER_* from the environment).  The path has no exchange step
    ("replicas only"): the process group is used for the barrier and the max over ranks only."""
    if world <= 1:
        return None
    import torch
    import torch.distributed as dist

    if backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device(device))
    else:
        dist.init_process_group(backend)
    return dist


def max_over_ranks(value, dist, device="cpu"):
    """The timed region of a multi-rank run is the slowest rank's."""
    if dist is None:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def time_oracle(P, budget_s=20.0):
    """cpu_baseline: the oracle as it stands, single thread, on a bounded sample (a few superiorized sweeps)."""
    from oracle.oracle import Oracle

    O = Oracle.from_problem(P)
    t0 = time.perf_counter()
    done = 0
    x, ell = P.x0, 0
    while True:
        R = O.superiorize(x, 1, P.N, P.beta0, P.a, lam=P.lam, ell0=ell)
        x, ell = R["x"], R["ell"]
        done += 1
        el = time.perf_counter() - t0
        if el >= budget_s or done >= P.n_sweeps or el + el / done > 1.5 * budget_s:
            break
    return done / el, done, el


def run_reference(args, rank, world):
    if rank != 0:
        return
    P = make_problem(args.workload)
    from oracle.oracle import Oracle

    O = Oracle.from_problem(P)
    sweeps_per_step = 1  # bounded sample: one superiorized sweep of the workload per step
    x, ell = P.x0, 0
    for _ in range(args.warmup):
        R = O.superiorize(x, sweeps_per_step, P.N, P.beta0, P.a, lam=P.lam, ell0=ell)
        x, ell = R["x"], R["ell"]
    t0 = time.perf_counter()
    for _ in range(args.steps):
        R = O.superiorize(x, sweeps_per_step, P.N, P.beta0, P.a, lam=P.lam, ell0=ell)
        x, ell = R["x"], R["ell"]
    el = time.perf_counter() - t0
    v = args.steps * sweeps_per_step / el
    sample = f"{sweeps_per_step} superiorized sweep(s) of the workload per step, continuing one run (sweeps 0..{args.steps + args.warmup - 1})"
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": WORKLOAD_TEXT.get(args.workload, args.workload), "m": P.m, "n": P.n, "nnz": P.nnz},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch

    import paper_2606_27086_b200 as sup
    from paper_2606_27086_b200.binding import create_from_problem

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (libsup has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    dist = dist_setup(world, "nccl", dev)

    if args.workload == "cfg5:all":
        return run_cfg5_all(args, dev)
    P = make_problem(args.workload)
    if args.sharded:
        return run_sharded(args, P, rank, world, local_rank, dev, dist)
    if args.block:  # BASELINE.json configs[2], second run: block-iterative with 16 interleaved angle blocks (A-14)
        import gen

        P = gen.interleaved_angle_blocks(P, 16)
    t0 = time.perf_counter()
    H = create_from_problem(P, dtype=sup.F32, device=dev)
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    S = P.n_sweeps
    x0 = torch.tensor(P.x0, dtype=torch.float32, device=dev)
    x = x0.clone()
    kw = dict(objective=P.objective, shape=P.shape, lam=P.lam, block=bool(args.block))

    def step():
        x.copy_(x0)
        sup.sup_superiorize(H, x, S, P.N, P.beta0, P.a, **kw)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    launches0 = H.launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = H.launches - launches0
    st = sup.sup_get_state(H)
    sampler.stop_flag = True
    ms = max_over_ranks(ms, dist, dev)
    value = world * args.steps * S / (ms * 1e-3)

    # ---- e2e: the C-ABI call with HOST buffers (pinned), H2D + D2H inside the timed region -------------------
    xh0 = torch.tensor(P.x0, dtype=torch.float32).pin_memory()
    xh = xh0.clone().pin_memory()
    for _ in range(2):
        xh.copy_(xh0)
        sup.sup_superiorize_host(H, xh, S, P.N, P.beta0, P.a, **kw)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        xh.copy_(xh0)
        sup.sup_superiorize_host(H, xh, S, P.N, P.beta0, P.a, **kw)  # synchronises
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dist, dev)
    e2e = world * args.steps * S / e2e_s
    checksum = float(xh.double().sum())

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the two product kernels, each timed alone with CUDA events on the library's stream ------
    peak, peak_src = load_peak()
    reps = 20
    xs = x0.clone()
    sup.sup_project_simultaneous(H, xs, 1.0, 3)  # a realistic iterate / y
    torch.cuda.synchronize()
    kern = {}
    bytes_fwd = 8 * P.nnz + 24 * P.m + 4 * P.n   # val+col, rowptr 8 + lb 4 + ub 4 + d 4 + y written 4, x read 4
    bytes_bwd = 8 * P.nnz + 24 * P.n + 4 * P.m   # val+idx, colptr 8 + x read 4 + lo 4 + hi 4 + x written 4, y read 4
    for name, fn, nbytes in (("k_fwd (S1+S2)", lambda: sup.sup_forward_violation(H, xs, sync_streams=False), bytes_fwd),
                             ("k_bwd (S3)", lambda: sup.sup_backproject_update(H, xs, 1.0, sync_streams=False), bytes_bwd)):
        for _ in range(3):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        H.stream.synchronize()
        a.record(H.stream)
        for _ in range(reps):
            fn()
        b.record(H.stream)
        H.stream.synchronize()
        t_ms = a.elapsed_time(b) / reps
        kern[name] = {"ms": t_ms, "algorithmic_bytes": nbytes, "gbs": nbytes / (t_ms * 1e-3) / 1e9}
    # unperturbed sweep (both kernels) for the share check
    H._check(sup.lib().sup_project_simultaneous(H.h, xs.data_ptr(), 1.0, 3))
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    H.stream.synchronize()
    a.record(H.stream)
    H._check(sup.lib().sup_project_simultaneous(H.h, xs.data_ptr(), 1.0, reps))
    b.record(H.stream)
    H.stream.synchronize()
    sweep_ms = a.elapsed_time(b) / reps
    # the same S sweeps WITHOUT perturbations, in the timed region's own protocol (from x0, graph replay, sustained clocks): what the
    # perturbation phases cost per sweep is superiorized_sweep_ms - basic_sweep_sustained_ms
    xb = x0.clone()
    for _ in range(2):
        xb.copy_(x0)
        sup.sup_superiorize(H, xb, S, 0, P.beta0, P.a, **kw)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for _ in range(args.steps):
        xb.copy_(x0)
        sup.sup_superiorize(H, xb, S, 0, P.beta0, P.a, **kw)
    b.record()
    torch.cuda.synchronize()
    basic_sustained_ms = a.elapsed_time(b) / (args.steps * S)
    dom = max(kern, key=lambda k: kern[k]["ms"])
    sup_ms = ms / (args.steps * S)
    roof = {"bound": "hbm", "kernel": dom, "achieved": kern[dom]["gbs"], "peak": peak, "unit": "GB/s", "frac": kern[dom]["gbs"] / peak,
            "traffic": None, "peak_source": peak_src, "frac_of_nominal_8000": kern[dom]["gbs"] / 8000.0,
            "kernels": kern, "timing_note": "each product kernel timed alone over 20 back-to-back launches (burst clocks); the sweeps below are "
                                            "sustained runs under the power cap",
            "basic_sweep_ms": sweep_ms,
            "basic_sweep_gbs": (bytes_fwd + bytes_bwd) / (sweep_ms * 1e-3) / 1e9,
            "basic_sweep_frac_of_nominal_8000": (bytes_fwd + bytes_bwd) / (sweep_ms * 1e-3) / 8e12,
            "basic_sweep_sustained_ms": basic_sustained_ms,
            "perturbation_ms_per_sweep": sup_ms - basic_sustained_ms,
            "superiorized_sweep_ms": sup_ms,
            "superiorized_sweep_gbs": (bytes_fwd + bytes_bwd) / (sup_ms * 1e-3) / 1e9,
            "superiorized_sweep_frac_of_nominal_8000": (bytes_fwd + bytes_bwd) / (sup_ms * 1e-3) / 8e12}
    tr = os.path.join(ROOT, "profiles", "traffic.csv")  # per-launch DRAM bytes from the committed ncu --set full capture
    if os.path.exists(tr):
        import csv

        for row in csv.DictReader(open(tr)):
            if row["workload"] == args.workload and row["kernel"] == dom and not args.block:
                roof["traffic"] = int(row["dram_bytes_per_launch"])
                roof["traffic_source"] = "committed ncu --set full capture, not measured in this run: profiles/" + row["source"]

    cpu_v, cpu_done, cpu_el = time_oracle(P, args.cpu_budget) if args.cpu_budget > 0 else (None, 0, 0.0)
    extra_cpu = {}
    if args.cpu_budget > 0:  # builder's CPU restatements: reported baselines, not the oracle and not the target
        from baseline.cpu_restatement import time_openmp, time_scipy

        v, dn, el = time_scipy(P, min(args.cpu_budget, 10.0))
        extra_cpu["cpu_baseline_scipy"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "builder's CPU restatement (scipy.sparse fp32 csr_matrix products + NumPy TV, the paper's CPU structure, PAPER.md:L249)",
                                           "sample": f"first {dn} superiorized sweeps of the same workload ({el:.1f} s)"}
        v, dn, el, thr = time_openmp(P, min(args.cpu_budget, 10.0))
        extra_cpu["cpu_baseline_openmp"] = {"value": v, "unit": UNIT, "cores": thr, "kind": "builder's CPU restatement (plain fp64 CSR loops in C, OpenMP row-parallel forward and transposed products, NumPy TV)",
                                            "sample": f"first {dn} superiorized sweeps of the same workload ({el:.1f} s, host has {os.cpu_count()} cores)"}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": WORKLOAD_TEXT.get(args.workload, args.workload), "name": P.name, "m": P.m, "n": P.n, "nnz": P.nnz,
                   "sweeps_per_step": S, "N": P.N, "beta0": P.beta0, "a": P.a, "lambda": P.lam, "objective": P.objective,
                   "l2_note": (f"A and A^T ({16 * P.nnz / 1e9:.2f} GB) are far larger than the 126 MB L2, so every sweep streams them from HBM; no flush needed"
                               if 16 * P.nnz > 4 * 126e6 else
                               f"A and A^T ({16 * P.nnz / 1e6:.1f} MB) fit the 126 MB L2 and are NOT flushed: launch/latency-bound workload, sweeps/s only, no HBM fraction is claimed for it"),
                   "sweep": "block-iterative, 16 interleaved angle blocks" if args.block else "simultaneous",
                   "parallelism": "replicas only" if world > 1 else "single GPU", "setup_s": setup_s,
                   "final_ell": st["ell"], "trials_per_step": st["n_trials"], "checksum_x": checksum},
        "roofline": roof,
        "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"first {cpu_done} superiorized sweeps of the same workload ({cpu_el:.1f} s, single thread, host has {os.cpu_count()} cores)"},
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": int(P.n * 4), "d2h_bytes_per_step": int(P.n * 4)},
        "gpu_launches": int(launches),
        "clocks": sampler.summary(),
    }
    line.update(extra_cpu)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_cfg5_all(args, dev):
    """BASELINE.json configs[4]: the whole throughput sweep, m = 2^16 .. 2^24 x k = 16 / 64 / 256, 20 sweeps with and without the
    1-D TV perturbation, sweeps/s and GB/s (B_sweep = 16 nnz + 28 m + 28 n) per point.  Inputs are generated on the device
    (gen/device.py, bit-identical to the host recipe).  Points with more than 2^28 stored entries: the oracle is NOT run; 4 096
    seeded rows of y = D c(x) are recomputed on the host in fp64 from regenerated rows, and x* must be a fixed point."""
    import numpy as np
    import torch

    import gen
    import paper_2606_27086_b200 as sup
    from gen.device import config5_on_device

    table = []
    free_b, total_b = torch.cuda.mem_get_info()
    for k in (16, 64, 256):
        for lg in range(16, 25):
            m, nnz = 1 << lg, (1 << lg) * k
            row = {"log2m": lg, "k": k, "nnz": nnz}
            need = 72 * nnz + (1 << 30)
            if nnz > 0xfffffffe or need > free_b:
                row["status"] = f"not run: needs ~{need / 1e9:.0f} GB with the explicit A^T (device has {total_b / 1e9:.0f} GB)"
                table.append(row)
                continue
            G = config5_on_device(lg, k, dev)
            H = sup.sup_create(G["rowptr"], G["col"], G["val"], G["lb"], G["ub"], G["lo"], G["hi"], None, dtype=sup.F32, n=G["n"], device=dev)
            # x* inside every slab and the box: a fixed point, bit for bit
            xs = G["x_true"].clone()
            sup.sup_project_simultaneous(H, xs, 1.0, 2)
            row["x_star_fixed"] = bool(torch.equal(xs, G["x_true"]))
            x = G["x0"].clone()

            def timed(fn, reps=2):
                fn()
                best = 1e30
                for _ in range(reps):
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    x.copy_(G["x0"])
                    torch.cuda.synchronize()
                    a.record()
                    fn()
                    b.record()
                    torch.cuda.synchronize()
                    best = min(best, a.elapsed_time(b))
                return best * 1e-3

            t_basic = timed(lambda: sup.sup_project_simultaneous(H, x, 1.0, 20))
            prox = [sup.sup_proximity(H, G["x0"], 0), sup.sup_proximity(H, x, 0)]
            t_tv = timed(lambda: sup.sup_superiorize(H, x, 20, 5, 1.0, 0.99, objective="tv1d"))
            bsweep = 16 * nnz + 28 * m + 28 * G["n"]
            row.update(status="ok", basic_sweeps_per_s=20 / t_basic, basic_gbs=bsweep * 20 / t_basic / 1e9, tv1d_sweeps_per_s=20 / t_tv,
                       tv1d_gbs=bsweep * 20 / t_tv / 1e9, proximity_x0=prox[0], proximity_after_20=prox[1],
                       regime="L2-resident" if 16 * nnz < 100e6 else "HBM stream, gathers from L2")
            if nnz > (1 << 28):  # oracle not run: fp64 spot check of 4096 rows of y = D c(x)
                x.copy_(G["x_true"] * 0.5)
                sup.sup_forward_violation(H, x)
                from paper_2606_27086_b200.binding import sup_get_derived

                y = sup_get_derived(H, 5)
                rng = np.random.default_rng(lg * 1000 + k)
                rows = np.unique(rng.integers(0, m, 4096))
                t = np.arange(k, dtype=np.uint64)[None, :]
                h = gen.workloads.hash3(gen.SEED0 + 5, rows.astype(np.uint64)[:, None], t)
                w = np.uint64(G["n"] // k)
                cols = (t * w + h % w).astype(np.int64)
                vals = (((h >> np.uint64(40)) + np.uint64(1)).astype(np.float64) / 2.0**24).astype(np.float32).astype(np.float64)
                xh = x.cpu().numpy().astype(np.float64)
                r = (vals * xh[cols]).sum(1)
                lbh, ubh = G["lb"][rows].cpu().numpy().astype(np.float64), G["ub"][rows].cpu().numpy().astype(np.float64)
                c = np.where(r > ubh, r - ubh, np.where(r < lbh, r - lbh, 0.0))
                want = (1.0 / m) / (vals * vals).sum(1) * c
                got = y[rows].cpu().numpy().astype(np.float64)
                err = np.abs(got - want) / np.maximum(np.abs(want), 1e-30)
                row["spot_check_rows"] = int(rows.size)
                row["spot_check_max_rel_err"] = float(err[np.abs(want) > 1e-12].max()) if np.any(np.abs(want) > 1e-12) else 0.0
                row["oracle"] = "not run (nnz > 2^28): fp64 spot check of seeded rows + fixed point + proximity decrease"
            table.append(row)
            print(json.dumps(row), file=sys.stderr, flush=True)
            sup.sup_destroy(H)
            del H, G, x, xs
            torch.cuda.empty_cache()
    line = {"metric": METRIC, "unit": UNIT, "n_gpus": 1, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[4]: hyperslab-projection throughput sweep, m = 2^16..2^24, n = m/2, k = 16/64/256, "
                                   "20 sweeps with and without the 1-D TV perturbation (N=5, a=0.99)"},
            "value": max((r.get("tv1d_sweeps_per_s", 0.0) for r in table), default=0.0), "table": table}
    print(json.dumps(line), flush=True)


def run_sharded(args, P, rank, world, local_rank, dev, dist):
    """Row blocks of A per rank, replica of x, one all-reduce per sweep: total work is fixed -> strong scaling.
    The sweeps are driven from Python (no CUDA graph across the collective), the perturbation phase is replicated."""
    import torch

    import paper_2606_27086_b200 as sup
    from paper_2606_27086_b200.sharded import ShardedSup

    group = dist.group.WORLD if dist is not None else None
    Sh = ShardedSup(P, rank, world, dtype=sup.F32, device=dev, group=group)
    S = P.n_sweeps
    x0 = torch.tensor(P.x0, dtype=torch.float32, device=dev)
    x = x0.clone()

    def step():
        x.copy_(x0)
        Sh.superiorize(x, S, P.N, P.beta0, P.a, lam=P.lam)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = Sh.H.launches
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1), dist, dev)
    if rank == 0:
        line = {"metric": METRIC, "value": args.steps * S / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": WORKLOAD_TEXT.get(args.workload, args.workload), "m": P.m, "n": P.n, "nnz": P.nnz, "sweeps_per_step": S,
                           "parallelism": f"rows of A sharded over {world} rank(s), replica of x, one all-reduce of {P.n * 4} bytes per sweep",
                           "rows_of_rank0": [int(Sh.cuts[0]), int(Sh.cuts[1])]},
                "gpu_launches": int(Sh.H.launches - launches0), "checksum_x": float(x.double().sum())}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--block", action="store_true", help="block-iterative sweeps, 16 interleaved angle blocks (CT workloads)")
    ap.add_argument("--sharded", action="store_true", help="row-sharded sweeps over the N ranks (one all-reduce of an n-vector per sweep; "
                                                           "strong scaling) instead of N replicas")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started without a launcher: become N ranks (one process per GPU) under torch.distributed.run, or fail loudly
        import torch

        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(29500 + os.getpid() % 2000), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={world} ranks")
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
