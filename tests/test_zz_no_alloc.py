"""sup_tv2d_value_static: the one entry point that allocates nothing (scratch in a static device array, include/sup.h), checked
against the existing path sup_objective (per-CTA partials in the handle's workspace) -- same value up to the summation order --
on two calls in a row that share the static scratch.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu

TD = {0: torch.float32, 1: torch.float64}
TOL = 1e-12  # fp64 terms and sums on both sides; only the summation order differs (the bar test_gpu_parity.py uses for fp64 scalars)


def _identity_handle(sup, n, dtype):
    rp, c = np.arange(n + 1, dtype=np.int64), np.arange(n, dtype=np.int32)
    one, zero = np.ones(n, np.float32), np.zeros(n, np.float32)
    return sup.sup_create(rp, c, one, zero, one, zero, one, None, dtype=dtype, n=n)


@pytest.mark.parametrize("dtype", [0, 1])
def test_static_entry_matches_the_existing_path_on_two_calls_in_a_row(dtype):
    import paper_2606_27086_b200 as sup

    rng = np.random.default_rng(41)
    # the second image has FEWER rows than the first: stale row sums of call 1 stay in the scratch behind it and must not be read
    shapes = [(700, 301), (93, 517)]
    xs = [torch.tensor(rng.uniform(0, 1, ny * nx), dtype=TD[dtype], device="cuda:0") for ny, nx in shapes]
    want = []
    for (ny, nx), x in zip(shapes, xs):
        H = _identity_handle(sup, ny * nx, dtype)
        want.append(sup.sup_objective(H, x, "tv2d", (ny, nx)))
        sup.sup_destroy(H)
    out = torch.zeros(2, dtype=torch.float64, device="cuda:0")
    # two calls back to back on one stream, no synchronisation in between, each into its own output slot
    for k, ((ny, nx), x) in enumerate(zip(shapes, xs)):
        sup.sup_tv2d_value_static(x, (ny, nx), out=out[k:k + 1], sync=False)
    got = out.cpu().numpy()
    for k in range(2):
        assert want[k] > 0 and abs(got[k] - want[k]) <= TOL * abs(want[k]), (k, got[k], want[k])
    # and once more in the other order, synchronising: the same bits as before (fixed summation order, shared scratch left clean)
    again = [sup.sup_tv2d_value_static(xs[1], shapes[1]), sup.sup_tv2d_value_static(xs[0], shapes[0])]
    assert again[0] == got[1] and again[1] == got[0]


def test_static_entry_edge_shapes_and_limits():
    import paper_2606_27086_b200 as sup
    from paper_2606_27086_b200.binding import STATIC_MAX_ROWS, SupError

    x = torch.rand(4096, dtype=torch.float32, device="cuda:0")
    assert sup.sup_tv2d_value_static(x, (1, 4096)) == 0.0 and sup.sup_tv2d_value_static(x, (4096, 1)) == 0.0  # no 2 x 2 neighbourhood
    # 2 x 2 by hand: one term sqrt((c - a)^2 + (b - a)^2)
    q = torch.tensor([1.0, 4.0, 5.0, 9.0], dtype=torch.float64, device="cuda:0")
    assert sup.sup_tv2d_value_static(q, (2, 2)) == pytest.approx(5.0, rel=1e-15)
    # the maximum number of rows is accepted, one more is refused before any launch, with a text that says why
    tall = torch.rand(STATIC_MAX_ROWS * 3, dtype=torch.float32, device="cuda:0")
    H = _identity_handle(sup, tall.numel(), 0)
    want = sup.sup_objective(H, tall, "tv2d", (STATIC_MAX_ROWS, 3))
    sup.sup_destroy(H)
    assert abs(sup.sup_tv2d_value_static(tall, (STATIC_MAX_ROWS, 3)) - want) <= TOL * want
    too_tall = torch.rand((STATIC_MAX_ROWS + 1) * 2, dtype=torch.float32, device="cuda:0")
    with pytest.raises(SupError, match="beyond the static scratch"):
        sup.sup_tv2d_value_static(too_tall, (STATIC_MAX_ROWS + 1, 2))
    with pytest.raises(SupError):
        sup.sup_tv2d_value_static(x, (0, 5))
