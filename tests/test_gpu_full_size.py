"""GPU parity at FULL size against the oracle's stored results (tests/golden/*.npz, written by tests/golden/make_goldens.py,
which imports only gen/ and oracle/): BASELINE.json configs[2] (512x512 low-dose CT, simultaneous and 16-block) and
configs[3] (IMRT, feasible and infeasible), in the launch configuration bench.py times (no overrides, CUDA graph).

Bars (north_star): fp32 x <= 1e-4 / fp64 <= 1e-10 relative L2, proximity and objective 1e-4, decisions and l exact
(A-13 for knife edges).  Three protocols, as in test_gpu_parity.py:
  basic      10 (5) unperturbed sweeps from x0, free-running                                             -- strict
  step-wise  ONE superiorized sweep from a state of the oracle's own run (x^k rounded to the handle's type, l_k, k)  -- strict
  free run   the first 10 (5) superiorized sweeps from x0 through the graph replay -- north_star's bars are applied and the
             outcome is REPORTED (met / not met); where the iteration is conditioning-limited (A-23) the assert is
             the documented looser bound, and DESIGN.md section 7 lists the case as not met.
"""
import json
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu

import gen  # noqa: E402

GOLD = os.path.join(os.path.dirname(__file__), "golden")
TD = {0: torch.float32, 1: torch.float64}
TOL = {0: 1e-4, 1: 1e-10}
KNIFE = {0: 1e-6, 1: 1e-12}
_cache = {}


def rel_l2(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a - b)


def load(name):
    if name not in _cache:
        G = dict(np.load(os.path.join(GOLD, name + ".npz")))
        meta = json.loads(str(G["meta"]))
        if name == "cfg3_full_simul":
            P = gen.config3_lowdose_ct()
        elif name == "cfg3_full_block":
            P = gen.interleaved_angle_blocks(gen.config3_lowdose_ct(), 16)
        else:
            P = gen.config4_imrt(infeasible=name.endswith("infeasible"))
        assert (P.m, P.n, P.nnz) == (meta["m"], meta["n"], meta["nnz"]), "the generator no longer produces the golden's problem"
        _cache.clear()  # one full-size problem in host memory at a time
        _cache[name] = (P, G, meta)
    return _cache[name]


def handle(P, dtype):
    from paper_2606_27086_b200.binding import create_from_problem

    return create_from_problem(P, dtype=dtype)


def run_gpu(H, P, x, cnt, ell, k, block, cap=1 << 16):
    import paper_2606_27086_b200 as sup

    dec = torch.zeros(cap, dtype=torch.int8, device="cuda:0")
    trace = torch.zeros((cnt, 4), dtype=torch.float64, device="cuda:0")
    sup.sup_superiorize(H, x, cnt, P.N, P.beta0, P.a, objective=P.objective, shape=P.shape, lam=P.lam, block=block, ell0=ell, k0=k,
                        trace=trace, decisions=dec, use_graph=True)
    st = sup.sup_get_state(H)
    assert st["fault"] == 0 and st["warn"] == 0 and st["n_decisions"] <= cap
    return st["ell"], dec[: st["n_decisions"]].cpu().numpy().copy(), trace.cpu().numpy()


def check_step(P, G, H, dtype, block, xs, ell, k, want_x, want_dec, want_mar, want_ell, want_trace, tag):
    """one superiorized sweep from a common state: everything strict"""
    x = torch.tensor(np.asarray(xs), dtype=TD[dtype], device="cuda:0")
    ell_g, dec, tr = run_gpu(H, P, x, 1, ell, k, block)
    if not (dec.size == want_dec.size and np.array_equal(dec, want_dec)):
        nmin = min(dec.size, want_dec.size)
        diff = np.flatnonzero(dec[:nmin] != want_dec[:nmin])
        first = int(diff[0]) if diff.size else nmin
        margin = want_mar[first] if first < want_mar.size else 0.0
        raise AssertionError(f"{tag}: decisions differ at trial {first}, oracle margin {margin:g} (knife edge below {KNIFE[dtype]:g})")
    assert ell_g == want_ell, (tag, ell_g, want_ell)
    err = rel_l2(x.cpu().numpy(), want_x)
    print(f"[full-size step-wise] {tag}: rel L2 {err:.3e} (bar {TOL[dtype]:g}), {dec.size} trials, l = {ell_g}")
    assert err <= TOL[dtype], (tag, err)
    for j, nm in ((0, "proximity"), (1, "objective")):
        assert abs(tr[0, j] - want_trace[j]) <= 1e-4 * abs(want_trace[j]) + 1e-300, (tag, nm, tr[0, j], want_trace[j])
    assert tr[0, 2] == want_trace[2] and tr[0, 3] == want_trace[3]


def full_size_case(name, dtype, S, kstep, block):
    import paper_2606_27086_b200 as sup

    P, G, meta = load(name)
    assert meta["sweeps"] == S and meta["step_ks"] == [kstep]
    H = handle(P, dtype)
    # ---- basic algorithm, free-running: strict ----
    x = torch.tensor(P.x0, dtype=TD[dtype], device="cuda:0")
    run = sup.sup_block_iterative if block else sup.sup_project_simultaneous
    run(H, x, P.lam, 1)
    e1 = rel_l2(x.cpu().numpy(), G["basic_x1"])
    run(H, x, P.lam, S - 1)
    eS = rel_l2(x.cpu().numpy(), G[f"basic_x{S}"])
    stored64 = f"basic_x{S}" in meta["f64_keys"]
    tolS = TOL[dtype] if (dtype == 0 or stored64) else 1e-6  # a golden stored as fp32 cannot certify 1e-10
    print(f"[full-size basic] {name} dtype={dtype}: sweep 1 {e1:.3e}, sweep {S} {eS:.3e} (bar {tolS:g})")
    assert e1 <= max(TOL[dtype], 1e-7) and eS <= tolS
    # ---- superiorized, step-wise from the oracle's own states: strict ----
    tr, dec, mar = G["sup_trace"], G["sup_decisions"], G["sup_margins"]
    n1 = int(tr[0, 2])
    if dtype == 0 or "sup_x1" in meta["f64_keys"]:
        check_step(P, G, H, dtype, block, P.x0, 0, 0, G["sup_x1"], dec[:n1], mar[:n1], int(tr[0, 3]), tr[0], f"{name} dtype={dtype} k=0")
    ell_k = int(tr[kstep - 1, 3])
    if dtype == 0:  # from fl32(x^k): the oracle's re-synchronised sweep
        xs = np.asarray(G[f"sup_x{kstep}"], np.float32)
        check_step(P, G, H, dtype, block, xs, ell_k, kstep, G[f"step{kstep}_x"], G[f"step{kstep}_decisions"], G[f"step{kstep}_margins"],
                   int(G[f"step{kstep}_ell"]), G[f"step{kstep}_trace"][0], f"{name} dtype=0 k={kstep}")
    elif f"sup_x{kstep}" in meta["f64_keys"]:  # fp64: x^k itself -> x^{k+1} of the free run
        nbefore = int(tr[:kstep, 2].sum())
        check_step(P, G, H, dtype, block, G[f"sup_x{kstep}"], ell_k, kstep, G[f"sup_x{kstep + 1}"], dec[nbefore:], mar[nbefore:],
                   int(tr[kstep, 3]), tr[kstep], f"{name} dtype=1 k={kstep}")
    # ---- superiorized, free run through the graph replay: north_star's bars applied, outcome reported ----
    x = torch.tensor(P.x0, dtype=TD[dtype], device="cuda:0")
    ell_g, gdec, gtr = run_gpu(H, P, x, S, 0, 0, block)
    same = gdec.size == dec.size and np.array_equal(gdec, dec)
    err = rel_l2(x.cpu().numpy(), G[f"sup_x{S}"])
    first = None
    if not same:
        nmin = min(gdec.size, dec.size)
        diff = np.flatnonzero(gdec[:nmin] != dec[:nmin])
        first = int(diff[0]) if diff.size else nmin
    knife = (not same) and first < mar.size and mar[first] < KNIFE[dtype]  # A-13: both outcomes are faithful executions
    met = (same or knife) and err <= TOL[dtype] and (dtype == 0 or f"sup_x{S}" in meta["f64_keys"])
    print(f"[full-size free run] {name} dtype={dtype}: sweep {S} rel L2 {err:.3e} (bar {TOL[dtype]:g}), decisions "
          f"{'identical' if same else f'differ from trial {first} (oracle margin {mar[first] if first < mar.size else 0:g})'}, "
          f"l {ell_g} vs {int(G['sup_ell'])}, prox {gtr[-1, 0]:.6e} vs {tr[-1, 0]:.6e}, f {gtr[-1, 1]:.6e} vs {tr[-1, 1]:.6e} "
          f"-> north_star bar {'MET' + (' (decision flip at a knife edge, A-13)' if knife else '') if met else 'NOT MET (A-23: conditioning-limited)'}")
    # whatever the amplification, the run must stay close and healthy: the documented looser bound
    assert err <= (5e-3 if dtype == 0 else 1e-6), (name, dtype, err)
    assert abs(gtr[-1, 0] - tr[-1, 0]) <= 1e-3 * abs(tr[-1, 0]) and abs(gtr[-1, 1] - tr[-1, 1]) <= 1e-2 * abs(tr[-1, 1]) + 1e-300


@pytest.mark.parametrize("dtype", [0, 1])
def test_config3_full_simultaneous_against_oracle_goldens(dtype):
    full_size_case("cfg3_full_simul", dtype, 10, 9, block=False)


def test_config3_full_block_iterative_against_oracle_goldens():
    full_size_case("cfg3_full_block", 0, 10, 9, block=True)


@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("variant", ["cfg4_full", "cfg4_full_infeasible"])
def test_config4_full_against_oracle_goldens(variant, dtype):
    full_size_case(variant, dtype, 5, 4, block=False)


def test_config3_full_back_to_back_kernels_equal_idle_device():
    """At the size bench.py times: 10 sweeps enqueued back to back (each product kernel a programmatic dependent of the one before)
    against the same 20 kernels with the device idle between any two -- bit-identical"""
    import paper_2606_27086_b200 as sup

    P, G, meta = load("cfg3_full_simul")
    H = handle(P, 0)
    xa = torch.tensor(P.x0, dtype=torch.float32, device="cuda:0")
    xb = xa.clone()
    sup.sup_project_simultaneous(H, xa, P.lam, 10)
    torch.cuda.synchronize()
    for _ in range(10):
        sup.sup_forward_violation(H, xb)
        torch.cuda.synchronize()
        sup.sup_backproject_update(H, xb, P.lam)
        torch.cuda.synchronize()
    assert torch.equal(xa, xb)
    assert rel_l2(xa.cpu().numpy(), G["basic_x10"]) <= 1e-4
