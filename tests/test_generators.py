"""Self-checks of the seeded workload generators (gen/): geometry only, no method arithmetic."""
import numpy as np
import pytest

import gen


def chord_in_square(theta, s, half):
    """length of {x cos + y sin = s} inside [-half, half)^2 by clipping the parametrised line."""
    c, sn = np.cos(theta), np.sin(theta)
    lo, hi = -1e9, 1e9
    for p0, d in ((s * c, -sn), (s * sn, c)):
        if abs(d) < 1e-15:
            if p0 < -half or p0 >= half:
                return 0.0
        else:
            a, b = (-half - p0) / d, (half - p0) / d
            lo, hi = max(lo, min(a, b)), min(hi, max(a, b))
    return max(0.0, hi - lo)


def test_ct_rows_sum_to_chord_and_canonical():
    npix, na, nb = 32, 24, 47
    rp, col, val = gen.ct_matrix(npix, na, nb)
    assert rp[0] == 0 and rp.size == na * nb + 1 and col.dtype == np.int32 and val.dtype == np.float32
    for r in range(na * nb):
        c = col[rp[r]:rp[r + 1]]
        assert (np.diff(c) > 0).all()  # sorted, distinct
        q, p = divmod(r, nb)
        th = 0.0 if q == 0 else q * np.pi / na
        ch = chord_in_square(th, p - (nb - 1) / 2, npix / 2) if 2 * q != na else chord_in_square(np.pi / 2, p - (nb - 1) / 2, npix / 2)
        assert val[rp[r]:rp[r + 1]].astype(np.float64).sum() == pytest.approx(ch, abs=2e-5)
    assert val.min() >= 1e-7 and val.max() <= np.sqrt(2) * (1 + 1e-6)
    assert col.min() >= 0 and col.max() < npix * npix


def test_ct_tiny_against_numerical_line_integral():
    npix, na, nb = 8, 5, 9
    rp, col, val = gen.ct_matrix(npix, na, nb)
    A = np.zeros((na * nb, npix * npix))
    for r in range(na * nb):
        A[r, col[rp[r]:rp[r + 1]]] = val[rp[r]:rp[r + 1]]
    t = (np.arange(200000) + 0.5) / 200000 * 24.0 - 12.0
    dt = 24.0 / 200000
    for q in range(na):
        th = q * np.pi / na
        for p in range(nb):
            s = p - 4.0
            x = s * np.cos(th) - t * np.sin(th)
            y = s * np.sin(th) + t * np.cos(th)
            jx, iy = np.floor(x + 4).astype(int), np.floor(y + 4).astype(int)
            ok = (jx >= 0) & (jx < 8) & (iy >= 0) & (iy < 8)
            num = np.bincount((iy * 8 + jx)[ok], minlength=64) * dt
            if q == 0:  # rays lie exactly on grid lines: half-open pixels -> the + side column (or nothing at the edge)
                expect = np.zeros(64)
                if 0 <= p < 8:
                    expect[np.arange(8) * 8 + p] = 1.0
                np.testing.assert_allclose(A[q * nb + p], expect, atol=1e-6)
            else:
                np.testing.assert_allclose(A[q * nb + p], num, atol=5e-4)


def test_ct_quarter_turn_symmetry():
    # angle q + na/2 is angle q rotated by 90 degrees: pixel (i,j) -> (j, n-1-i) maps rows with s -> s (odd bins, centred)
    npix, na, nb = 16, 8, 23
    rp, col, val = gen.ct_matrix(npix, na, nb)
    A = np.zeros((na * nb, npix, npix))
    for r in range(na * nb):
        c = col[rp[r]:rp[r + 1]]
        A[r, c // npix, c % npix] = val[rp[r]:rp[r + 1]]
    for q in range(1, na // 2):  # generic angles (q = 0 has the half-open edge rule)
        for p in range(nb):
            a = A[q * nb + p]
            b = A[(q + na // 2) * nb + p]
            # rotating the image by +90 deg sends pixel (i, j) to (j, n-1-i): b[j, n-1-i] = a[i, j]
            np.testing.assert_allclose(b, np.rot90(a, -1), atol=2e-6)


def test_segments_rows_sum_to_length():
    P = gen.config2_crosswell(n_grid=32, n_src=8, n_rcv=8)
    seg = P.meta["segments"]
    L = np.hypot(seg[:, 2] - seg[:, 0], seg[:, 3] - seg[:, 1])
    rs = np.asarray(P.scipy().sum(axis=1)).ravel()
    np.testing.assert_allclose(rs, L, atol=2e-5)
    assert (np.diff(P.rowptr) >= 32).all()
    assert (P.lb < P.ub).all() and P.x0.min() == pytest.approx(0.1)


def test_imrt_entries_follow_the_stated_formula():
    P = gen.config4_imrt(scale=0.2)
    gx, gy, gz = P.meta["grid"]
    h, nb, bs, sig = P.meta["h"], P.meta["nb"], P.meta["bs"], P.meta["sigma"]
    vox = P.meta["vox"]
    A = P.scipy().tocsc()
    colmax = np.asarray(A.max(axis=0).todense()).ravel()
    rng = np.random.default_rng(0)
    rows = rng.choice(np.flatnonzero(np.diff(P.rowptr) > 0), 20, replace=False)
    for r in rows:
        lin = vox[r]
        x, y, z = lin % gx, (lin // gx) % gy, lin // (gx * gy)
        p = np.array([(x - (gx - 1) / 2) * h, (y - (gy - 1) / 2) * h, (z - (gz - 1) / 2) * h])
        for k in range(P.rowptr[r], P.rowptr[r + 1]):
            c = P.col[k]
            b, v, u = c // (nb * nb), (c // nb) % nb, c % nb
            phi = P.meta["phis"][b]
            depth = 240.0 + p[0] * np.cos(phi) + p[1] * np.sin(phi)
            lu = (-p[0] * np.sin(phi) + p[1] * np.cos(phi)) - (u - (nb - 1) / 2) * bs
            lv = p[2] - (v - (nb - 1) / 2) * bs
            expect = np.exp(-0.005 * depth) * np.exp(-(lu * lu + lv * lv) / (2 * sig * sig))
            assert P.val[k] == pytest.approx(expect, rel=1e-6)
            assert P.val[k] >= 1e-3 * colmax[c] * (1 - 1e-6)
    assert (P.lb[np.isfinite(P.lb)] == 57.0).all() and set(np.unique(P.ub)) <= {20.0, 30.0, 64.2, 66.0}.union({np.float32(64.2)})
    assert P.dose[3] == P.m


def test_imrt_infeasible_variant_duplicates_overlap_rows():
    P = gen.config4_imrt(scale=0.5, infeasible=True)
    md = P.dose[3]
    assert P.m > md, "the overlap PTV/OAR1 must contain voxels at this scale"
    # every duplicated row repeats a PTV row's entries and carries the OAR bound
    assert (P.ub[md:] == 20.0).all() and np.isinf(P.lb[md:]).all()
    key = lambda r: (P.col[P.rowptr[r]:P.rowptr[r + 1]].tobytes(), P.val[P.rowptr[r]:P.rowptr[r + 1]].tobytes())
    ptv_rows = {key(r) for r in np.flatnonzero(P.lb[:md] == 57.0)}
    assert all(key(r) in ptv_rows for r in range(md, P.m))
    # D_body is A without the duplicates
    assert np.array_equal(P.dose[0], P.rowptr[: md + 1]) and np.array_equal(P.dose[1], P.col[: P.rowptr[md]])


def test_config5_structure_and_feasible_point():
    for k in (16, 64):
        P = gen.config5_sweep_point(12, k)
        assert P.m == 4096 and P.n == 2048 and P.nnz == 4096 * k
        c = P.col.reshape(P.m, k)
        assert (np.diff(c, axis=1) > 0).all() and c.min() >= 0 and c.max() < P.n
        assert P.val.min() > 0 and P.val.max() <= 1
        r = P.scipy() @ P.x_true.astype(np.float64)
        assert (r > P.lb).all() and (r < P.ub).all()
        assert (P.ub - P.lb).max() <= 0.2 + 1e-4
    # the counter hash is reproducible and seed-dependent
    a = gen.random_csr(1024, 16, 5)
    b = gen.random_csr(1024, 16, 5)
    c2 = gen.random_csr(1024, 16, 6)
    assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2]) and not np.array_equal(a[1], c2[1])


def test_config1_and_3_recipes_small():
    P = gen.config1_tiny_ct()
    assert (P.m, P.n) == (8190, 4096) and P.objective == "tv2d" and P.shape == (64, 64)
    assert np.allclose(P.ub - P.lb, 4 * P.meta["sigma"], rtol=1e-5)
    assert 0 <= P.x_true.min() and P.x_true.max() <= 1
    Q = gen.config3_lowdose_ct(n_pix=32, n_angles=16, n_bins=47)
    assert np.isinf(Q.hi).all() and (Q.lo == 0).all() and (Q.lb < Q.ub).all()
    B = gen.interleaved_angle_blocks(Q, 4)
    assert B.block_rowptr.tolist() == [0, 4 * 47, 8 * 47, 12 * 47, 16 * 47]
    perm = B.meta["row_perm"]
    A, Ab = Q.scipy().toarray(), B.scipy().toarray()
    assert np.array_equal(Ab, A[perm]) and np.array_equal(B.lb, Q.lb[perm])
    assert set((perm[: 4 * 47] // 47) % 4) == {0}
