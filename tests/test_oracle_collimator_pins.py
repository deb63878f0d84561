"""Pins of the collimator rotation of the oracle (reading G25): the fluence map is
resampled (bilinear, zero outside) on its own grid after a rotation about the central axis, before the projection."""
import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_2512_18863_b200 import workloads as W


def square_case(n=15, **kw):
    wl = W.tiny(seed=81, flu=(n, n), flu_d=3.0, **kw)
    return wl, Oracle(wl.grid, wl.model, wl.density)


def test_quarter_turns_are_exact_permutations_and_zero_is_the_identity():
    """On a square map with square pixels a rotation by a multiple of 90 degrees maps pixel centres onto pixel centres:
    numpy.rot90 / flips (independent routine).  Memory is [v][u]; +90 degrees takes the +u axis onto the +v axis."""
    wl, orc = square_case()
    M = np.random.Generator(np.random.PCG64(81)).uniform(0, 1, orc.flu_shape)
    assert np.array_equal(orc.rotate_map(0.0, M), M)
    assert np.allclose(orc.rotate_map(180.0, M), M[::-1, ::-1], rtol=0, atol=1e-12)
    # Phirot(u,v) = Phi(R(-90)(u,v)) = Phi(v, -u): rot[b][a] = M[(n-1)-a][b]
    want = M[::-1, :].T
    assert np.allclose(orc.rotate_map(90.0, M), want, rtol=0, atol=1e-12)
    assert np.allclose(orc.rotate_map(-90.0, orc.rotate_map(90.0, M)), M, rtol=0, atol=1e-12)
    # sign convention on a single spot: a spot at +u moves to +v under +90 degrees
    spot = np.zeros(orc.flu_shape)
    spot[7, 11] = 1.0                                     # (u, v) = (+4 px, 0)
    r = orc.rotate_map(90.0, spot)
    assert r[11, 7] == pytest.approx(1.0, abs=1e-12) and r.sum() == pytest.approx(1.0, abs=1e-12)


def test_small_angle_moves_the_centroid_like_a_rotation_and_conserves_the_sum():
    wl, orc = square_case(n=41)
    a = np.arange(41) - 20.0
    U, V = np.meshgrid(a, a)                              # [v][u]
    blob = np.exp(-((U - 8.0) ** 2 + (V - 3.0) ** 2) / 8.0)
    for ang in (7.0, -23.0, 41.0):
        r = orc.rotate_map(ang, blob)
        cu, cv = (r * U).sum() / r.sum(), (r * V).sum() / r.sum()
        c, s = np.cos(np.radians(ang)), np.sin(np.radians(ang))
        assert cu == pytest.approx(c * 8.0 - s * 3.0, abs=0.02) and cv == pytest.approx(s * 8.0 + c * 3.0, abs=0.02)
        assert r.sum() == pytest.approx(blob.sum(), rel=2e-3)


def test_rotation_adjoint_identity():
    wl = W.tiny(seed=82, flu=(17, 13), flu_d=2.5)
    orc = Oracle(wl.grid, wl.model, wl.density)
    rng = np.random.Generator(np.random.PCG64(82))
    x, y = rng.standard_normal(orc.flu_shape), rng.standard_normal(orc.flu_shape)
    for ang in (0.0, 33.0, 90.0, -147.0):
        lhs = float((orc.rotate_map(ang, x) * y).sum())
        rhs = float((x * orc.rotate_map(ang, y, transpose=True)).sum())
        assert lhs == pytest.approx(rhs, rel=1e-12, abs=1e-12)


def test_collimator_90_equals_the_field_with_swapped_axes():
    """An open rectangular field (leaves retracted): jaws (x = +-12, y = +-21) at collimator 90 give the dose of jaws
    (x = +-21, y = +-12) at collimator 0 — square map, square pixels, no penumbra / off-axis asymmetry between the axes."""
    wl, orc = square_case(n=21, nx=30, ny=28, nz=30, spacing=3.0, n_cp=1, kernel_size=5, head_scatter=False, gantry=[20.0])
    wl.model.update(fwhm_mlc_mm=0.0, fwhm_jaw_mm=0.0)
    wl.grid["iso"] = (0.0, 0.0, 0.0)
    orc = Oracle(wl.grid, wl.model, wl.density)
    lv = np.zeros((1, 2, wl.model["n_pairs"]))
    lv[:, 0], lv[:, 1] = -100.0, 100.0
    d90 = orc.dose_coll(lv, [[-12.0, 12.0, -21.0, 21.0]], wl.gantry_deg, [90.0], wl.mu)
    d0 = orc.dose_coll(lv, [[-21.0, 21.0, -12.0, 12.0]], wl.gantry_deg, [0.0], wl.mu)
    assert d0.max() > 0 and np.abs(d90 - d0).max() <= 1e-10 * d0.max()
    assert np.array_equal(d0, orc.dose(lv, [[-21.0, 21.0, -12.0, 12.0]], wl.gantry_deg, wl.mu))        # angle 0 == the plain path


def test_gradients_with_collimator_vs_finite_differences():
    wl = W.tiny(seed=83, n_cp=2, nx=22, ny=20, nz=10, kernel_size=5, flu=(16, 12), head_scatter=False)
    orc = Oracle(wl.grid, wl.model, wl.density)
    rng = np.random.Generator(np.random.PCG64(83))
    g = rng.standard_normal(orc.dose_shape).astype(np.float32)
    lv, jw, mu = wl.leaves.astype(np.float64), wl.jaws.astype(np.float64), wl.mu.astype(np.float64)
    coll = np.array([25.0, -70.0])
    dl, dj, dm = orc.dose_backward_coll(lv, jw, wl.gantry_deg, coll, mu, g)
    L = lambda l, j, m: float((orc.dose_coll(l, j, wl.gantry_deg, coll, m) * g).sum())
    h = 1e-4
    for (b, bank, i) in ((0, 0, 2), (1, 1, 3)):
        p, q = lv.copy(), lv.copy()
        p[b, bank, i] += h; q[b, bank, i] -= h
        assert dl[b, bank, i] == pytest.approx((L(p, jw, mu) - L(q, jw, mu)) / (2 * h), rel=1e-6, abs=1e-10)
    for (b, e) in ((0, 1), (1, 2)):
        p, q = jw.copy(), jw.copy()
        p[b, e] += h; q[b, e] -= h
        assert dj[b, e] == pytest.approx((L(lv, p, mu) - L(lv, q, mu)) / (2 * h), rel=1e-6, abs=1e-10)
    p, q = mu.copy(), mu.copy()
    p[0] += h; q[0] -= h
    assert dm[0] == pytest.approx((L(lv, jw, p) - L(lv, jw, q)) / (2 * h), rel=1e-8)
