"""Host-side logic of the N > 1 path of bench.py on CPU (gloo, world size 2): the path is "replicas only"
(DESIGN.md section 8), so what there is to test is the rendezvous from the environment, the barrier, the
max-over-ranks of the timed region, and that the reference arm runs on rank 0 alone."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench

    dist = bench.dist_setup(world, "gloo")
    dist.barrier()
    got = bench.max_over_ranks(10.0 + 5.0 * rank, dist)  # rank 1 is the slow one
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, got))


def test_max_over_ranks_gloo_world2():
    mp = pytest.importorskip("torch.multiprocessing")
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == {0: 15.0, 1: 15.0}


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.dist_setup(1, "gloo") is None
    assert bench.max_over_ranks(3.5, None) == 3.5


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
           "--warmup", "1", "--workload", "cfg1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] == 0


def test_gpus_flag_means_n_ranks_or_fails_loudly():
    """`bench.py --gpus N` without a launcher must itself become N ranks -- here, with no CUDA device, it must refuse instead of
    silently timing one GPU; under a launcher the world size must equal --gpus."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2"], capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "only 0 CUDA device(s) visible" in (r.stdout + r.stderr)
    env = dict(os.environ, WORLD_SIZE="4", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2"], capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode != 0 and "WORLD_SIZE=4" in (r.stdout + r.stderr)


def _shard_worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import numpy as np
    import torch
    import torch.distributed as dist

    import gen
    from paper_2606_27086_b200.sharded import partition_rows, row_block

    dist.init_process_group("gloo")
    P = gen.config1_tiny_ct(n_pix=24, n_angles=20, n_bins=35)
    cuts = partition_rows(P.rowptr, world)
    r0, r1 = int(cuts[rank]), int(cuts[rank + 1])
    rp, col, val, lb, ub = row_block(P, r0, r1)
    lb, ub = lb.astype(np.float64), ub.astype(np.float64)
    # host stand-in for the two kernels of a block (the CUDA path cannot run here): the block's share of A^T D c(x)
    x = np.linspace(0.0, 1.0, P.n)
    rho = np.add.reduceat(val.astype(np.float64) ** 2, rp[:-1][np.diff(rp) > 0]) if val.size else np.zeros(0)
    u = np.zeros(P.n)
    k = 0
    for i in range(r1 - r0):
        s, e = rp[i], rp[i + 1]
        if e > s:
            a = val[s:e].astype(np.float64)
            r = float(a @ x[col[s:e]])
            c = r - ub[i] if r > ub[i] else (r - lb[i] if r < lb[i] else 0.0)
            u[col[s:e]] += a * ((1.0 / P.m) / rho[k] * c)
            k += 1
    t = torch.from_numpy(u)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    dist.destroy_process_group()
    out.put((rank, cuts.tolist(), t.numpy().copy()))


def test_row_sharding_partition_and_allreduce_gloo_world2():
    """contiguous row blocks balanced by nonzeros, one all-reduce of an n-vector per sweep: the blocks' shares of
    A^T D c(x), summed over the ranks, are the unsharded back-projection (host arithmetic stands in for the kernels here; the
    kernels themselves are checked on the GPU by test_row_sharded_sweep_matches_single_handle)."""
    import numpy as np

    mp = pytest.importorskip("torch.multiprocessing")
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    ps = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = [q.get(timeout=180) for _ in ps]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    sys.path.insert(0, ROOT)
    import gen
    from oracle.oracle import Oracle

    P = gen.config1_tiny_ct(n_pix=24, n_angles=20, n_bins=35)
    cuts = res[0][1]
    assert cuts[0] == 0 and cuts[-1] == P.m and cuts == res[1][1]
    nnz_block = [int(P.rowptr[cuts[g + 1]] - P.rowptr[cuts[g]]) for g in range(2)]
    assert abs(nnz_block[0] - nnz_block[1]) <= 2 * int(np.diff(P.rowptr).max())
    x = np.linspace(0.0, 1.0, P.n)
    O = Oracle(P.m, P.n, P.rowptr, P.col, P.val, P.lb, P.ub, np.full(P.n, -np.inf), np.full(P.n, np.inf))
    want = x - O.sweep(x, 1.0)  # u = A^T D c(x)
    for _, _, u in res:
        np.testing.assert_allclose(u, want, rtol=1e-10, atol=1e-14)
