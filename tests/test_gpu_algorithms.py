"""GPU parity of the SURVEY.md 8(f) rows against the oracle: DROP and EMR (Table A.5), the paper's stopping
rule (L217-223, L239-243; A-25), f_Mean (Eq. 21) and the 3-D TV objective (A-27).  Same bars as test_gpu_parity.py."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu

import gen  # noqa: E402
from oracle.oracle import Oracle  # noqa: E402

TD = {0: torch.float32, 1: torch.float64}
TOL = {0: 1e-4, 1: 1e-10}


def rel_l2(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a - b)


def _sup():
    import paper_2606_27086_b200 as sup

    return sup


def equality_ct(n_pix=40, n_angles=36, n_bins=57, noise=0.01, seed=3):
    """a CT-shaped EQUALITY problem (lb = ub = b), the case Table A.5 prints"""
    P = gen.config1_tiny_ct(n_pix=n_pix, n_angles=n_angles, n_bins=n_bins, n_sweeps=12, N=3)
    rng = np.random.default_rng(seed)
    b = P.scipy() @ P.x_true.astype(np.float64)
    b = (b + noise * b.max() * rng.normal(size=P.m)).astype(np.float32)
    P.lb, P.ub = b.copy(), b.copy()
    P.name = "ct_equality"
    return P


def handle(P, dtype):
    from paper_2606_27086_b200.binding import create_from_problem

    return create_from_problem(P, dtype=dtype, blocks=False)


def xdev(x, dtype):
    return torch.tensor(np.asarray(x), dtype=TD[dtype], device="cuda:0")


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("which", ["equality", "slabs", "cfg2"])
def test_drop_and_emr_sweeps(which, dtype):
    sup = _sup()
    P = equality_ct() if which == "equality" else (gen.config1_tiny_ct(n_pix=37, n_angles=23, n_bins=61) if which == "slabs" else gen.config2_crosswell())
    H = handle(P, dtype)
    O = Oracle.from_problem(P)
    # DROP, with two relaxations
    for lam in (1.0, 1.7):
        x = xdev(P.x0, dtype)
        xo = P.x0.astype(np.float64)
        for s in (1, 7):
            sup.sup_project_drop(H, x, lam, s)
            xo = O.drop_sweep(xo, lam, s)
            assert rel_l2(x.cpu().numpy(), xo) <= TOL[dtype], (which, "drop", lam, s)
    # EMR: the iterate and the relaxation factor of the last sweep
    x = xdev(P.x0, dtype)
    xo = P.x0.astype(np.float64)
    for s in range(8):
        sup.sup_project_emr(H, x, 1)
        xo, t = O.emr_sweep(xo, 1, return_step=True)
        st = sup.sup_get_state(H)
        assert abs(st["step"] - t) <= (1e-4 if dtype == 0 else 1e-10) * abs(t), (which, s, st["step"], t)
        assert rel_l2(x.cpu().numpy(), xo) <= TOL[dtype], (which, "emr", s)
    # the sweeps leave the library in a consistent state: a plain simultaneous sweep afterwards still matches
    sup.sup_project_simultaneous(H, x, 1.0, 2)
    assert rel_l2(x.cpu().numpy(), O.sweep(xo, 1.0, 2)) <= TOL[dtype]


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("alg", ["drop", "emr"])
def test_superiorized_drop_and_emr_stepwise(alg, dtype):
    """TV-superiorized DROP / EMR (the paper's CT experiment runs EMR this way, L342): one sweep at a time from the oracle's state"""
    sup = _sup()
    P = equality_ct()
    H = handle(P, dtype)
    O = Oracle.from_problem(P)
    lam = 1.9 if alg == "drop" else 1.0
    x_ref, ell = P.x0.astype(np.float64), 0
    for k in range(8):
        xs = np.asarray(x_ref, np.float32 if dtype == 0 else np.float64).astype(np.float64)
        R = O.run(xs, 1, N=P.N, beta0=P.beta0, a=0.9, lam=lam, algorithm=alg, ell0=ell, k0=k)
        x = xdev(xs, dtype)
        dec = torch.zeros(4096, dtype=torch.int8, device="cuda:0")
        sup.sup_superiorize(H, x, 1, P.N, P.beta0, 0.9, objective="tv2d", shape=P.shape, lam=lam, algorithm=alg, ell0=ell, k0=k, decisions=dec)
        st = sup.sup_get_state(H)
        assert st["ell"] == R["ell"] and np.array_equal(dec[: st["n_decisions"]].cpu().numpy(), R["decisions"]), (alg, k)
        assert rel_l2(x.cpu().numpy(), R["x"]) <= TOL[dtype], (alg, dtype, k)
        x_ref, ell = R["x"], R["ell"]
    # and the graph replay of several sweeps stays within the final-sweep bar
    x = xdev(P.x0, dtype)
    sup.sup_superiorize(H, x, 8, P.N, P.beta0, 0.9, objective="tv2d", shape=P.shape, lam=lam, algorithm=alg)
    R = O.run(P.x0, 8, N=P.N, beta0=P.beta0, a=0.9, lam=lam, algorithm=alg)
    assert rel_l2(x.cpu().numpy(), R["x"]) <= (1e-3 if dtype == 0 else 1e-9)


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("case", ["basic", "tv", "block_tv", "emr_tv", "never"])
def test_stopping_rule_stops_where_the_oracle_stops(case, dtype):
    """Oracle and GPU stop after the same sweep for the same reason; x is the iterate the rule was met at; a rule that never
    fires leaves the fixed-length run bit-identical; the trace (proximity, objective per sweep) agrees."""
    sup = _sup()
    base = gen.config1_tiny_ct(n_pix=32, n_angles=40, n_bins=47, n_sweeps=60, N=3)
    P = gen.interleaved_angle_blocks(base, 8) if case == "block_tv" else base
    from paper_2606_27086_b200.binding import create_from_problem

    H = create_from_problem(P, dtype=dtype)
    O = Oracle.from_problem(P)
    pert = case != "basic"
    alg = {"block_tv": "block", "emr_tv": "emr"}.get(case, "sim")
    N = P.N if pert else 0
    K = 60
    # thresholds chosen from the oracle's own fixed-length trace so that the rule fires somewhere in the middle of the run
    ref = O.run(P.x0, K, N=N, beta0=P.beta0, a=0.9, lam=P.lam, algorithm=alg, kind=P.objective if pert else "none")
    Pk = 2.0 * ref["trace"][:, 0]
    fk = ref["trace"][:, 1]
    dP = np.abs(np.diff(Pk)) / np.maximum(1.0, Pk[:-1])
    df = np.abs(np.diff(fk)) / np.maximum(1.0, fk[:-1])
    if case == "never":
        stop = dict(prox_tol=-1.0, dprox_tol=0.0, n_consec=5, dobj_tol=0.0)
    else:
        # every threshold sits in the (geometric) middle of a gap of the oracle's own values, so that neither side decides a
        # comparison by its last bits (the knife-edge rule of A-13 applied to the stopping test)
        gap = lambda v, q: float(np.sqrt(np.sort(v)[q] * np.sort(v)[q + 1]))
        below = Pk[Pk < Pk[25]]
        stop = dict(prox_tol=float(np.sqrt(Pk[25] * below.max())) if below.size else float(Pk[25]) * 0.999,
                    dprox_tol=gap(dP, len(dP) // 2), n_consec=3, dobj_tol=gap(df, int(0.8 * len(df))) if pert else 1.0)
    R = O.run(P.x0, K, N=N, beta0=P.beta0, a=0.9, lam=P.lam, algorithm=alg, kind=P.objective if pert else "none", stop=stop)
    x = xdev(P.x0, dtype)
    trace = torch.zeros((K, 4), dtype=torch.float64, device="cuda:0")
    sup.sup_superiorize(H, x, K, N, P.beta0, 0.9, objective=P.objective if pert else None, shape=P.shape, lam=P.lam, block=case == "block_tv",
                        algorithm=alg, stop=stop, trace=trace)
    st = sup.sup_get_state(H)
    print(f"[stopping] {case} dtype={dtype}: oracle stops after {R['n_done']} (reason {R['stop_reason']}), GPU after {st['n_done']} (reason {st['stop_reason']})")
    assert st["n_done"] == R["n_done"] and st["stop_reason"] == R["stop_reason"], (case, st, R["n_done"], R["stop_reason"])
    if case != "never":
        assert 0 < R["n_done"] < K, "the thresholds of this test must make the rule fire inside the run"
    tol = TOL[dtype] if R["n_done"] <= 12 else (1e-3 if dtype == 0 else 1e-8)
    assert rel_l2(x.cpu().numpy(), R["x"]) <= tol
    tr = trace.cpu().numpy()[: R["n_done"]]
    np.testing.assert_allclose(tr[:, 0], R["trace"][:, 0], rtol=1e-3 if dtype == 0 else 1e-7)
    if pert:
        np.testing.assert_allclose(tr[:, 1], R["trace"][:, 1], rtol=1e-3 if dtype == 0 else 1e-7)
    assert np.array_equal(tr[:, 3], R["trace"][:, 3])
    if case == "never":
        x2 = xdev(P.x0, dtype)
        sup.sup_superiorize(H, x2, K, N, P.beta0, 0.9, objective=P.objective, shape=P.shape, lam=P.lam)
        assert torch.equal(x, x2)


@pytest.mark.parametrize("dtype", [0, 1])
def test_mean_objective(dtype):
    """f_Mean (Eq. 21) over an organ-at-risk of the reduced IMRT case: value, phase (every first trial accepted), Algorithm 1"""
    sup = _sup()
    P = gen.config4_imrt(scale=0.17)
    rp, c, v, md = P.dose
    vox_is_oar = (P.ub[:md] <= 30.5)  # rows bounded by 20 or 30 Gy: the two OARs
    rows = np.flatnonzero(vox_is_oar)
    counts = np.diff(rp)[rows]
    rp_s = np.zeros(rows.size + 1, np.int64)
    np.cumsum(counts, out=rp_s[1:])
    idx = np.repeat(rp[:-1][rows] - rp_s[:-1], counts) + np.arange(rp_s[-1], dtype=np.int64)
    DS = (rp_s, c[idx], v[idx], rows.size)
    assert rows.size >= 5
    H = sup.sup_create(P.rowptr, P.col, P.val, P.lb, P.ub, P.lo, P.hi, None, dtype=dtype, n=P.n)
    sup.sup_set_dose_matrix(H, DS[0], DS[1], DS[2])
    O = Oracle(P.m, P.n, P.rowptr, P.col, P.val, P.lb, P.ub, P.lo, P.hi, dose=DS, objective="mean")
    rng = np.random.default_rng(5)
    xs = rng.uniform(0.5, 1.5, P.n).astype(np.float32)
    x = xdev(xs, dtype)
    assert abs(sup.sup_objective(H, x, "mean") - O.objective_value(xs.astype(np.float64))) <= (1e-5 if dtype == 0 else 1e-12) * abs(O.objective_value(xs.astype(np.float64)))
    ell = sup.sup_perturb_mean(H, x, 4, 0.5, 0.9, 2)
    R = O.perturb(xs.astype(np.float64), 2, 4, 0.5, 0.9)
    st = sup.sup_get_state(H)
    assert ell == R["ell"] == 6 and st["n_trials"] == 4 and list(R["decisions"]) == [1, 1, 1, 1]
    assert rel_l2(x.cpu().numpy(), R["x"]) <= (1e-6 if dtype == 0 else 1e-13)
    assert abs(st["f"] - R["fx"]) <= (1e-5 if dtype == 0 else 1e-12) * abs(R["fx"])
    # Algorithm 1 with the mean objective, step-wise
    x_ref, ell = P.x0.astype(np.float64), 0
    for k in range(6):
        xs64 = np.asarray(x_ref, np.float32 if dtype == 0 else np.float64).astype(np.float64)
        R = O.run(xs64, 1, N=3, beta0=1.0, a=0.95, ell0=ell, k0=k)
        xg = xdev(xs64, dtype)
        sup.sup_superiorize(H, xg, 1, 3, 1.0, 0.95, objective="mean", ell0=ell, k0=k)
        assert sup.sup_get_state(H)["ell"] == R["ell"]
        assert rel_l2(xg.cpu().numpy(), R["x"]) <= TOL[dtype], k
        x_ref, ell = R["x"], R["ell"]


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("shape", [(6, 9, 40), (5, 8, 32), (1, 7, 11), (9, 1, 13), (3, 4, 1), (17, 19, 23)])
def test_tv3d_objective_and_phase(shape, dtype):
    sup = _sup()
    n = int(np.prod(shape))
    rng = np.random.default_rng(8)
    eye_rp = np.arange(n + 1, dtype=np.int64)
    eye_c = np.arange(n, dtype=np.int32)
    H = sup.sup_create(eye_rp, eye_c, np.ones(n, np.float32), np.zeros(n, np.float32), np.ones(n, np.float32), np.zeros(n, np.float32),
                       np.ones(n, np.float32), None, dtype=dtype, n=n)
    O = Oracle(n, n, eye_rp, eye_c, np.ones(n), np.zeros(n), np.ones(n), np.zeros(n), np.ones(n), objective="tv3d", shape=shape)
    xs = rng.uniform(0, 1, n).astype(np.float32)
    x = xdev(xs, dtype)
    fo = O.objective_value(xs.astype(np.float64))
    fg = sup.sup_objective(H, x, "tv3d", shape)
    assert abs(fg - fo) <= (1e-6 if dtype == 0 else 1e-12) * abs(fo) + (0 if fo else 1e-300)
    ell = 1
    xo = xs.astype(np.float64)
    for phase in range(3):
        ell_g = sup.sup_perturb_tv(H, x, shape, 3, 0.4, 0.8, ell)
        R = O.perturb(xo, ell, 3, 0.4, 0.8)
        st = sup.sup_get_state(H)
        assert ell_g == R["ell"] and st["n_trials"] == R["trials"], (shape, phase, ell_g, R["ell"], R["margins"].min() if R["margins"].size else None)
        assert rel_l2(x.cpu().numpy(), R["x"]) <= (1e-5 if dtype == 0 else 1e-13)
        assert abs(st["f"] - R["fx"]) <= (1e-5 if dtype == 0 else 1e-12) * abs(R["fx"]) + 1e-300
        xo, ell = R["x"], ell_g
    # Algorithm 1 over a box-only feasibility problem with the 3-D objective
    x = xdev(xs, dtype)
    sup.sup_superiorize(H, x, 4, 2, 0.4, 0.8, objective="tv3d", shape=shape)
    R = O.run(xs.astype(np.float64), 4, N=2, beta0=0.4, a=0.8)
    assert sup.sup_get_state(H)["ell"] == R["ell"]
    assert rel_l2(x.cpu().numpy(), R["x"]) <= TOL[dtype]


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("world", [2, 3])
def test_row_sharded_sweep_matches_single_handle(world, dtype):
    """SURVEY.md 8(e) on the real kernels, emulated on one GPU (the blocks run one after the other, nothing waits on anything):
    every block's share u_g = W_g A_g^T y_g summed = the unsharded back-projection; sharded superiorized sweeps against the
    single-handle run (summation order differs: tolerance 1e-6 / 1e-12 per sweep) and against the oracle at the usual bars."""
    sup = _sup()
    from paper_2606_27086_b200.sharded import ShardedSup

    P = gen.config1_tiny_ct(n_pix=40, n_angles=36, n_bins=57, n_sweeps=8, N=3)
    shards = [ShardedSup(P, g, world, dtype=dtype) for g in range(world)]
    assert sum(s.share for s in shards) == pytest.approx(1.0, rel=1e-12)
    H = handle(P, dtype)
    O = Oracle.from_problem(P)
    x_ref = xdev(P.x0, dtype)
    ell_ref = 0
    for k in range(8):
        xs = x_ref.clone()  # both start every sweep from the same state (A-23: the TV iteration amplifies roundings)
        # single handle: perturbation phase + sweep
        ell = sup.sup_perturb_tv(shards[0].H, xs, P.shape, P.N, P.beta0, P.a, ell_ref)
        ell_ref = sup.sup_perturb_tv(H, x_ref, P.shape, P.N, P.beta0, P.a, ell_ref)
        assert ell == ell_ref and torch.equal(xs, x_ref)  # the replicated perturbation phase is bit-identical
        sup.sup_project_simultaneous(H, x_ref, P.lam, 1)
        # sharded: per-block shares, "all-reduce" by hand, identical update
        u = torch.zeros_like(xs)
        for s in shards:
            u += s.partial(xs)
        sup.sup_apply_update(shards[0].H, xs, u, P.lam)
        assert rel_l2(xs.cpu().numpy(), x_ref.cpu().numpy()) <= (1e-6 if dtype == 0 else 1e-12), k
    # the sharded driver on its own (world = 1 group-less shards would skip the reduction, so drive the blocks by hand) vs the oracle
    xs, ell = xdev(P.x0, dtype), 0
    for k in range(8):
        ell = sup.sup_perturb_tv(shards[0].H, xs, P.shape, P.N, P.beta0, P.a, ell)
        u = torch.zeros_like(xs)
        for s in shards:
            u += s.partial(xs)
        sup.sup_apply_update(shards[0].H, xs, u, P.lam)
    R = O.superiorize(P.x0, 8, P.N, P.beta0, P.a, lam=P.lam)
    assert ell == R["ell"]
    assert rel_l2(xs.cpu().numpy(), R["x"]) <= (1e-3 if dtype == 0 else 1e-9)


@pytest.mark.parametrize("lg,k", [(12, 16), (13, 64), (14, 256)])
def test_device_generator_is_bit_identical(lg, k):
    """gen/device.py (the config-5 generator for points too large for the host) against gen.config5_sweep_point"""
    from gen.device import config5_on_device

    P = gen.config5_sweep_point(lg, k)
    G = config5_on_device(lg, k)
    assert np.array_equal(G["rowptr"].cpu().numpy(), P.rowptr) and np.array_equal(G["col"].cpu().numpy(), P.col)
    assert np.array_equal(G["val"].cpu().numpy(), P.val) and np.array_equal(G["x_true"].cpu().numpy(), P.x_true)
    assert np.array_equal(G["lb"].cpu().numpy(), P.lb) and np.array_equal(G["ub"].cpu().numpy(), P.ub)


def test_more_than_2_31_stored_entries():
    """64-bit nnz: m = 2^23 rows x k = 256 = 2^31 stored entries (row pointers int64, 32-bit unsigned ranks in the transpose):
    x* is a fixed point, the proximity decreases, seeded rows of y agree with an fp64 recomputation."""
    sup = _sup()
    from gen.device import config5_on_device
    from paper_2606_27086_b200.binding import sup_get_derived

    free_b, _ = torch.cuda.mem_get_info()
    lg, k = 23, 256
    if free_b < 72 * (1 << lg) * k + (2 << 30):
        pytest.skip("not enough device memory for the 2^31-entry point")
    G = config5_on_device(lg, k)
    m, n = G["m"], G["n"]
    H = sup.sup_create(G["rowptr"], G["col"], G["val"], G["lb"], G["ub"], G["lo"], G["hi"], None, dtype=0, n=n)
    xs = G["x_true"].clone()
    sup.sup_project_simultaneous(H, xs, 1.0, 1)
    assert torch.equal(xs, G["x_true"])
    x = G["x0"].clone()
    p0 = sup.sup_proximity(H, x, 0)
    sup.sup_project_simultaneous(H, x, 1.0, 2)
    p2 = sup.sup_proximity(H, x, 0)
    assert p2 < p0
    sup.sup_forward_violation(H, x)
    y = sup_get_derived(H, 5)
    rng = np.random.default_rng(1)
    rows = np.unique(np.concatenate([rng.integers(0, m, 2000), [0, m - 1, m // 2]]))
    t = np.arange(k, dtype=np.uint64)[None, :]
    h = gen.workloads.hash3(gen.SEED0 + 5, rows.astype(np.uint64)[:, None], t)
    w = np.uint64(n // k)
    cols = (t * w + h % w).astype(np.int64)
    vals = (((h >> np.uint64(40)) + np.uint64(1)).astype(np.float64) / 2.0**24).astype(np.float32).astype(np.float64)
    xh = x.cpu().numpy().astype(np.float64)
    r = (vals * xh[cols]).sum(1)
    lbh, ubh = G["lb"][rows].cpu().numpy().astype(np.float64), G["ub"][rows].cpu().numpy().astype(np.float64)
    c = np.where(r > ubh, r - ubh, np.where(r < lbh, r - lbh, 0.0))
    want = (1.0 / m) / (vals * vals).sum(1) * c
    got = y[rows].cpu().numpy().astype(np.float64)
    big = np.abs(c) > 1e-3
    assert big.sum() > 100
    np.testing.assert_allclose(got[big], want[big], rtol=2e-3)  # fp32 row dots of 256 terms against a violation of >= 1e-3


# ---- Eq. 11: the subgradient-projection step size (SUP_RULE_ADAPTIVE, reading A-30) ----------------------
def _identity_handle(sup, n, dtype):
    rp, c = np.arange(n + 1, dtype=np.int64), np.arange(n, dtype=np.int32)
    one, zero = np.ones(n, np.float32), np.zeros(n, np.float32)
    H = sup.sup_create(rp, c, one, zero, one, zero, one, None, dtype=dtype, n=n)
    return H, (n, n, rp, c, np.ones(n), np.zeros(n), np.ones(n), np.zeros(n), np.ones(n))


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("kind,shape", [("tv2d", (37, 91)), ("tv2d", (130, 70)), ("tv1d", (5000,)), ("tv3d", (6, 9, 40))])
def test_adaptive_phase_tv(kind, shape, dtype):
    sup = _sup()
    n = int(np.prod(shape))
    H, oargs = _identity_handle(sup, n, dtype)
    O = Oracle(*oargs, objective=kind, shape=shape if kind != "tv1d" else None)
    xs = np.random.default_rng(17).uniform(0, 1, n).astype(np.float32)
    f0 = O.objective_value(xs.astype(np.float64))
    sh = None if kind == "tv1d" else shape
    ptol, ftol = (2e-6, 1e-5) if dtype == 0 else (1e-13, 1e-12)
    for N in (1, 3):
        # above the reference: N steps of Eq. 11
        x = xdev(xs, dtype)
        fr = sup.sup_perturb_adaptive(H, x, kind, N, 0.9 * f0, 0.5, shape=sh)
        R = O.perturb_adaptive(xs.astype(np.float64), N, 0.9 * f0, 0.5)
        st = sup.sup_get_state(H)
        assert st["n_trials"] == R["steps"] == N and st["n_decisions"] == N and fr == R["f_ref"] == 0.9 * f0
        err = rel_l2(x.cpu().numpy(), R["x"])
        assert err <= ptol, (kind, shape, N, err)
        # at / below the reference: beta = 0, x untouched bit for bit, the reference moves to shrink * f(x)
        x = xdev(xs, dtype)
        fr = sup.sup_perturb_adaptive(H, x, kind, N, 2.0 * f0, 0.25, shape=sh)
        assert torch.equal(x, xdev(xs, dtype)) and sup.sup_get_state(H)["n_trials"] == 0
        assert abs(fr - 0.25 * f0) <= ftol * f0
    # a constant image has a zero gradient: no step although f = 0 > f_ref
    x = torch.full((n,), 0.5, dtype=TD[dtype], device="cuda:0")
    fr = sup.sup_perturb_adaptive(H, x, kind, 2, -1.0, 0.5, shape=sh)
    assert fr == -1.0 and bool((x == 0.5).all()) and sup.sup_get_state(H)["n_trials"] == 0


@pytest.mark.parametrize("dtype", [0, 1])
def test_adaptive_phase_dose_and_argument_errors(dtype):
    sup = _sup()
    P = gen.config4_imrt(scale=0.17)
    H = handle(P, dtype)
    O = Oracle.from_problem(P)
    xs = np.random.default_rng(3).uniform(0.5, 1.5, P.n).astype(np.float32)
    f0 = O.objective_value(xs.astype(np.float64), "dose")
    for N in (1, 3):
        x = xdev(xs, dtype)
        fr = sup.sup_perturb_adaptive(H, x, "dose", N, 0.8 * f0, 0.5)
        R = O.perturb_adaptive(xs.astype(np.float64), N, 0.8 * f0, 0.5, kind="dose")
        st = sup.sup_get_state(H)
        assert st["n_trials"] == R["steps"] == N and fr == 0.8 * f0
        err = rel_l2(x.cpu().numpy(), R["x"])
        assert err <= (2e-6 if dtype == 0 else 1e-12), (N, err)
    x = xdev(xs, dtype)
    fr = sup.sup_perturb_adaptive(H, x, "dose", 2, 1.5 * f0, 0.5)
    assert torch.equal(x, xdev(xs, dtype)) and abs(fr - 0.5 * f0) <= (1e-5 if dtype == 0 else 1e-12) * f0
    # arguments
    with pytest.raises(Exception):
        sup.sup_perturb_adaptive(H, x, "mean", 1, 0.0, 0.5)
    with pytest.raises(Exception):
        sup.sup_perturb_adaptive(H, x, "dose", 1, 0.0, 0.0)
    with pytest.raises(Exception):
        sup.sup_perturb_adaptive(H, x, "dose", 1, float("nan"), 0.5)
    with pytest.raises(Exception):
        sup.sup_superiorize(H, x, 2, 2, 1.0, 0.9, objective="dose", adaptive=dict(f_ref=0.0, shrink=0.5), n_restart=5)


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("which", ["cfg1", "cfg4"])
def test_adaptive_rule_inside_algorithm_1(which, dtype):
    """Eq. 10 with Eq. 11's step size: step-wise from the oracle's own states (strict), then a free run through the graph replay
    (step pattern identical, x within the free-run bound of A-23)"""
    sup = _sup()
    P = gen.config1_tiny_ct() if which == "cfg1" else gen.config4_imrt(scale=0.17)
    H = handle(P, dtype)
    O = Oracle.from_problem(P)
    kw = dict(objective=P.objective, shape=P.shape, lam=P.lam)
    f0 = O.objective_value(np.asarray(P.x0, np.float64))
    x_ref = np.asarray(P.x0, np.float64)
    if f0 == 0.0:  # x0 = 0: one basic sweep gives a start with f > 0
        x_ref = O.sweep(x_ref, P.lam)
        f0 = O.objective_value(x_ref)
    fr, shrink, N, S = 0.7 * f0, 0.6, 2, 8
    x_start = np.asarray(x_ref, np.float32 if dtype == 0 else np.float64).astype(np.float64)
    took = 0
    for k in range(S):
        xs64 = np.asarray(x_ref, np.float32 if dtype == 0 else np.float64).astype(np.float64)
        R = O.run(xs64, 1, N=N, lam=P.lam, adaptive=dict(f_ref=fr, shrink=shrink))
        xg = xdev(xs64, dtype)
        sup.sup_superiorize(H, xg, 1, N, 1.0, 0.9, adaptive=dict(f_ref=fr, shrink=shrink), **kw)
        st = sup.sup_get_state(H)
        assert st["n_trials"] == int(R["trace"][0, 2]) and st["ell"] == 0, (k, st, R["trace"])
        if R["f_ref"] == fr:
            assert st["f_ref"] == fr
        else:
            assert abs(st["f_ref"] - R["f_ref"]) <= (1e-5 if dtype == 0 else 1e-12) * abs(R["f_ref"])
        err = rel_l2(xg.cpu().numpy(), R["x"])
        assert err <= TOL[dtype], (which, k, err)
        took += int(R["trace"][0, 2])
        x_ref, fr = R["x"], R["f_ref"]
    assert 0 < took  # some steps were taken, and (below) the reference moved at least once in the free run
    # free run, CUDA graph
    fr0 = 0.7 * f0
    R = O.run(x_start, S, N=N, lam=P.lam, adaptive=dict(f_ref=fr0, shrink=shrink))
    xg = xdev(x_start, dtype)
    dec = torch.zeros(4 * S * N, dtype=torch.int8, device="cuda:0")
    sup.sup_superiorize(H, xg, S, N, 1.0, 0.9, adaptive=dict(f_ref=fr0, shrink=shrink), decisions=dec, use_graph=True, **kw)
    st = sup.sup_get_state(H)
    gdec = dec[: st["n_decisions"]].cpu().numpy()
    err = rel_l2(xg.cpu().numpy(), R["x"])
    print(f"[adaptive free run] {which} dtype={dtype}: rel L2 {err:.3e}, steps {gdec.sum()} vs {R['decisions'].sum()}, f_ref {st['f_ref']:.6e} vs {R['f_ref']:.6e}")
    assert st["n_decisions"] == S * N == R["decisions"].size
    if np.array_equal(gdec, R["decisions"]):
        assert err <= (5e-3 if dtype == 0 else 1e-8)
        assert abs(st["f_ref"] - R["f_ref"]) <= (1e-3 if dtype == 0 else 1e-9) * abs(R["f_ref"])


# ---- dose objective: the Gram-matrix path (sup_gram.cu) and the matrix-pass path are the same mathematics --------------------------
@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("mode", [0, 1])
def test_dose_phase_and_algorithm_1_in_both_dose_modes(mode, dtype):
    """mode 0: f = x^T (D^T D) x with G = D^T D built at sup_set_dose_matrix; mode 1: passes over D and D^T.  Each against the oracle
    (phase: trials, l, x, f; Algorithm 1 step-wise), and the Gram matrix itself against a dense fp64 product"""
    sup = _sup()
    P = gen.config4_imrt(scale=0.17)
    H = handle(P, dtype)
    sup.sup_set_dose_mode(H, mode)
    O = Oracle.from_problem(P)
    rng = np.random.default_rng(2)
    xs = rng.uniform(0.5, 1.5, P.n).astype(np.float32)
    x = xdev(xs, dtype)
    ell, xo = 3, xs.astype(np.float64)
    for phase in range(3):
        ell_g = sup.sup_perturb_dose(H, x, 4, P.beta0, 0.9, ell)
        st = sup.sup_get_state(H)
        R = O.perturb(xo, ell, 4, P.beta0, 0.9, kind="dose")
        xo = R["x"]
        assert ell_g == R["ell"] and st["n_trials"] == R["trials"], (phase, ell_g, R["ell"])
        assert rel_l2(x.cpu().numpy(), xo) <= (1e-5 if dtype == 0 else 1e-12), phase
        assert abs(st["f"] - R["fx"]) <= (1e-5 if dtype == 0 else 1e-11) * abs(R["fx"]), phase
        ell = ell_g
    # Algorithm 1, step-wise from the oracle's own states
    x_ref, ell = np.asarray(P.x0, np.float64), 0
    for k in range(6):
        xs64 = np.asarray(x_ref, np.float32 if dtype == 0 else np.float64).astype(np.float64)
        R = O.run(xs64, 1, N=P.N, beta0=P.beta0, a=P.a, lam=P.lam, ell0=ell, k0=k)
        xg = xdev(xs64, dtype)
        sup.sup_superiorize(H, xg, 1, P.N, P.beta0, P.a, objective="dose", lam=P.lam, ell0=ell, k0=k)
        assert sup.sup_get_state(H)["ell"] == R["ell"], k
        assert rel_l2(xg.cpu().numpy(), R["x"]) <= TOL[dtype], k
        x_ref, ell = R["x"], R["ell"]
    # free run through the graph: bit-identical to direct launches
    xa, xb = xdev(P.x0, dtype), xdev(P.x0, dtype)
    sup.sup_superiorize(H, xa, 7, P.N, P.beta0, P.a, objective="dose", lam=P.lam, use_graph=True)
    sup.sup_superiorize(H, xb, 7, P.N, P.beta0, P.a, objective="dose", lam=P.lam, use_graph=False)
    assert torch.equal(xa, xb)


def test_gram_matrix_is_dT_d():
    """G x and x^T G x of the Gram path against a dense fp64 restatement, through the public calls: one phase with a step so small
    that x does not move (beta0 tiny) reports f(x) = x^T G x; odd n (row padding) and rows longer than 64 entries included"""
    sup = _sup()
    rng = np.random.default_rng(11)
    md, n = 700, 77  # n not a multiple of 4 or 32; n^2 <= 2 nnz holds
    Dd = rng.uniform(0, 1, (md, n)) * (rng.random((md, n)) < 0.9)  # ~69 entries per row: the > 64 branch of the build kernel runs
    Dd[5] = 0.0  # an empty row
    rp = np.zeros(md + 1, np.int64)
    cols, vals = [], []
    for i in range(md):
        nz = np.flatnonzero(Dd[i])
        cols.append(nz)
        vals.append(Dd[i, nz])
        rp[i + 1] = rp[i] + nz.size
    c, v = np.concatenate(cols).astype(np.int32), np.concatenate(vals)
    assert n * n <= 2 * rp[-1] and np.diff(rp).max() > 64
    eye_rp, eye_c = np.arange(n + 1, dtype=np.int64), np.arange(n, dtype=np.int32)
    for dtype in (0, 1):
        H = sup.sup_create(eye_rp, eye_c, np.ones(n, np.float32), np.zeros(n, np.float32), np.full(n, 9.0, np.float32), np.zeros(n, np.float32),
                           np.full(n, 9.0, np.float32), None, dtype=dtype, n=n)
        sup.sup_set_dose_matrix(H, rp, c, v.astype(np.float32))
        D32 = Dd.astype(np.float32).astype(np.float64)
        G = D32.T @ D32
        xs = rng.uniform(0.5, 1.5, n).astype(np.float32)
        x = xdev(xs, dtype)
        sup.sup_perturb_dose(H, x, 1, 1e-30, 0.5, 0)
        st = sup.sup_get_state(H)
        f = xs.astype(np.float64) @ G @ xs.astype(np.float64)
        assert abs(st["f"] - f) <= (2e-6 if dtype == 0 else 1e-12) * f
        # one real step: x - c g with g = 2 G x, c = beta0 / ||g||
        x = xdev(xs, dtype)
        sup.sup_perturb_dose(H, x, 1, 0.01, 0.5, 0)
        g = 2 * G @ xs.astype(np.float64)
        want = xs.astype(np.float64) - 0.01 * g / np.linalg.norm(g)
        assert rel_l2(x.cpu().numpy(), want) <= (2e-7 if dtype == 0 else 1e-13)
        # an x that is not 16-byte aligned takes the kernel variant that stages the vector in shared memory: same bits
        buf = torch.zeros(n + 1, dtype=TD[dtype], device="cuda:0")
        xm = buf[1:]
        xm.copy_(xdev(xs, dtype))
        assert xm.data_ptr() % 16 != 0
        sup.sup_perturb_dose(H, xm, 1, 0.01, 0.5, 0)
        assert torch.equal(xm, x)


# ---- TV2D perturbation phase: the cluster kernel for small images (sup_perturb_small.cu) and the grid kernel ----------------------------
@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("shape", [(8, 8), (9, 37), (64, 64), (13, 1), (8, 512), (100, 300), (128, 256), (130, 256), (7, 40), (1, 64)])
def test_tv2d_phase_in_both_perturb_modes(shape, mode, dtype):
    """mode 0 sends images of >= 8 rows and <= 4096 pixels per row block to the cluster kernel ((130, 256), (7, 40) and (1, 64) are not
    eligible and take the grid kernel in both modes); mode 1 is the grid kernel.  Each against the oracle: trial sequence and l exact,
    x and f within the phase tolerances; power law (both policies), restarts and the adaptive rule"""
    sup = _sup()
    ny, nx = shape
    n = ny * nx
    H, oargs = _identity_handle(sup, n, dtype)
    sup.sup_set_perturb_mode(H, mode)
    O = Oracle(*oargs, objective="tv2d", shape=shape)
    rng = np.random.default_rng(ny * 1000 + nx)
    xs = (0.5 + 0.3 * np.sin(np.arange(n) * 0.37) + 0.05 * rng.normal(size=n)).astype(np.float32)
    ptol, ftol = (1e-5, 1e-4) if dtype == 0 else (1e-13, 1e-12)  # fp32: x and g are rounded to the storage type at every step (north_star: objective 1e-4)
    # power law: beta0 large enough that the first trials are rejected
    x = xdev(xs, dtype)
    xo, ell = xs.astype(np.float64), 2
    for phase in range(2):
        dec = torch.zeros(4096, dtype=torch.int8, device="cuda:0")
        ell_g = sup.sup_perturb_tv(H, x, shape, 4, 3.0, 0.8, ell)
        st = sup.sup_get_state(H)
        R = O.perturb(xo, ell, 4, 3.0, 0.8)
        xo = R["x"]
        assert ell_g == R["ell"] and st["n_trials"] == R["trials"], (shape, mode, phase, ell_g, R["ell"], R["margins"].min() if R["margins"].size else None)
        assert rel_l2(x.cpu().numpy(), xo) <= ptol, (shape, mode, phase)
        assert abs(st["f"] - R["fx"]) <= ftol * max(1.0, abs(R["fx"]))
        ell = ell_g
    # Algorithm 1 with the literal per-sweep policy and with restarts, decisions logged (needs a feasibility operator: identity rows)
    for kwargs in (dict(policy=sup.PER_SWEEP), dict(n_restart=2)):
        xg = xdev(xs, dtype)
        dec = torch.zeros(1 << 14, dtype=torch.int8, device="cuda:0")
        sup.sup_superiorize(H, xg, 5, 3, 1.5, 0.7, objective="tv2d", shape=shape, lam=1.0, decisions=dec, use_graph=True, **kwargs)
        st = sup.sup_get_state(H)
        if "policy" in kwargs:
            R = O.superiorize(xs.astype(np.float64), 5, 3, 1.5, 0.7, lam=1.0, policy=kwargs["policy"])
        else:
            R = O.superiorize(xs.astype(np.float64), 5, 3, 1.5, 0.7, lam=1.0, n_restart=2)
        gdec = dec[: st["n_decisions"]].cpu().numpy()
        if np.array_equal(gdec, R["decisions"]):
            assert st["ell"] == R["ell"]
            assert rel_l2(xg.cpu().numpy(), R["x"]) <= (1e-4 if dtype == 0 else 1e-10)
        else:  # a flipped accept test must be a knife edge (A-13)
            nmin = min(gdec.size, R["decisions"].size)
            first = int(np.flatnonzero(gdec[:nmin] != R["decisions"][:nmin])[0]) if nmin and (gdec[:nmin] != R["decisions"][:nmin]).any() else nmin
            assert first < R["margins"].size and R["margins"][first] < (1e-6 if dtype == 0 else 1e-12), (shape, mode, kwargs, first)
    # Eq. 11
    f0 = O.objective_value(xs.astype(np.float64))
    if f0 > 0:
        x = xdev(xs, dtype)
        fr = sup.sup_perturb_adaptive(H, x, "tv2d", 3, 0.9 * f0, 0.5, shape=shape)
        R = O.perturb_adaptive(xs.astype(np.float64), 3, 0.9 * f0, 0.5)
        assert sup.sup_get_state(H)["n_trials"] == R["steps"] and fr == R["f_ref"]
        assert rel_l2(x.cpu().numpy(), R["x"]) <= (2e-6 if dtype == 0 else 1e-13)
        x = xdev(xs, dtype)
        fr = sup.sup_perturb_adaptive(H, x, "tv2d", 2, 2.0 * f0, 0.25, shape=shape)
        assert torch.equal(x, xdev(xs, dtype)) and abs(fr - 0.25 * f0) <= ftol * f0


def test_cluster_and_grid_perturbation_kernels_take_the_same_decisions():
    """config 1 (64 x 64) through Algorithm 1 with both kernels: identical decision logs and l, x equal to rounding"""
    sup = _sup()
    P = gen.config1_tiny_ct()
    out = []
    for mode in (0, 1):
        H = handle(P, 0)
        sup.sup_set_perturb_mode(H, mode)
        x = xdev(P.x0, 0)
        dec = torch.zeros(1 << 14, dtype=torch.int8, device="cuda:0")
        sup.sup_superiorize(H, x, 12, P.N, P.beta0, P.a, objective="tv2d", shape=P.shape, lam=P.lam, decisions=dec)
        st = sup.sup_get_state(H)
        out.append((st["ell"], dec[: st["n_decisions"]].cpu().numpy().copy(), x.cpu().numpy().copy()))
    assert out[0][0] == out[1][0] and np.array_equal(out[0][1], out[1][1])
    assert rel_l2(out[0][2], out[1][2]) <= 1e-5
