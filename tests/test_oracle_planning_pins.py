"""Pins of the planning-loop part of the oracle: the Eq. 1-3 projection and its transposed
Jacobian, the Eq. 10 / quadratic objective, jaw tracking and the normalised-gradient step, checked against what the
paper and the mathematics fix (closed forms, invariants, finite differences, an independent numpy routine)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2512_18863_b200 import workloads as W

LIM = O.plan_limits(0.5, 96.0, 2.0, 100.0, 120.0, 0.1)


def random_params(seed, n_cp=7, n_pairs=11, spread=130.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    leaves = rng.uniform(-spread, spread, size=(n_cp, 2, n_pairs))          # unordered, beyond the travel range
    jaws = rng.uniform(-spread, spread, size=(n_cp, 4))
    mu = rng.uniform(-1.0, 3.0, size=n_cp)
    return leaves, jaws, mu


def test_projection_matches_eq_1_2_written_out():
    """Eq. 1-2 in plain numpy on every pair; Eq. 3's clamp on MU."""
    lv, jw, mu = random_params(1)
    pl, pj, pm = O.validate(LIM, lv, jw, mu)
    def proj(pa, pb, wmin, F):
        c, w = 0.5 * (pa + pb), pb - pa
        w = np.maximum(w, wmin)
        c = np.clip(c, -F, F)
        return c - 0.5 * w, c + 0.5 * w
    a, b = proj(lv[:, 0], lv[:, 1], 0.5, 96.0)
    assert np.array_equal(pl[:, 0], a) and np.array_equal(pl[:, 1], b)
    a, b = proj(jw[:, 0], jw[:, 1], 2.0, 100.0)
    assert np.array_equal(pj[:, 0], a) and np.array_equal(pj[:, 1], b)
    a, b = proj(jw[:, 2], jw[:, 3], 2.0, 120.0)
    assert np.array_equal(pj[:, 2], a) and np.array_equal(pj[:, 3], b)
    assert np.array_equal(pm, np.maximum(mu, 0.1))


def test_projection_is_feasible_and_idempotent():
    lv, jw, mu = random_params(2, n_cp=40)
    pl, pj, pm = O.validate(LIM, lv, jw, mu)
    assert (pl[:, 1] - pl[:, 0] >= 0.5 - 1e-12).all() and (np.abs(0.5 * (pl[:, 0] + pl[:, 1])) <= 96.0 + 1e-12).all()
    assert (pj[:, 1] - pj[:, 0] >= 2.0 - 1e-12).all() and (pj[:, 3] - pj[:, 2] >= 2.0 - 1e-12).all()
    assert (pm >= 0.1).all()
    ql, qj, qm = O.validate(LIM, pl, pj, pm)
    assert np.allclose(ql, pl, rtol=0, atol=1e-12) and np.allclose(qj, pj, rtol=0, atol=1e-12) and np.array_equal(qm, pm)
    # a feasible point is left alone exactly
    fl = np.stack([np.full((3, 5), -10.0), np.full((3, 5), 12.0)], axis=1)
    fj = np.tile([-20.0, 20.0, -30.0, 30.0], (3, 1))
    fm = np.full(3, 2.0)
    gl, gj, gm = O.validate(LIM, fl, fj, fm)
    assert np.array_equal(gl, fl) and np.array_equal(gj, fj) and np.array_equal(gm, fm)


def test_eq3_minimum_mu():
    """Eq. 3: eps = D_min * dphi / phidot_max; e.g. 0.6 MU/s * 2 deg / (6 deg/s) = 0.2 MU."""
    assert O.mu_epsilon(0.6, 2.0, 6.0) == pytest.approx(0.2, abs=1e-15)


def test_projection_jacobian_transpose_vs_finite_differences():
    """Away from the kinks (w = w_min, |c| = F, MU = eps) the map is linear in a neighbourhood, so central differences
    are exact to rounding; the transpose is checked through <J v, y> = <v, J^T y>."""
    lv, jw, mu = random_params(3)
    rng = np.random.Generator(np.random.PCG64(33))
    v = [rng.standard_normal(a.shape) for a in (lv, jw, mu)]
    y = [rng.standard_normal(a.shape) for a in (lv, jw, mu)]
    h = 1e-6
    plus = O.validate(LIM, lv + h * v[0], jw + h * v[1], mu + h * v[2])
    minus = O.validate(LIM, lv - h * v[0], jw - h * v[1], mu - h * v[2])
    Jv = [(p - m) / (2 * h) for p, m in zip(plus, minus)]
    JTy = O.validate_adjoint(LIM, lv, jw, mu, *y)
    lhs = sum(float((a * b).sum()) for a, b in zip(Jv, y))
    rhs = sum(float((a * b).sum()) for a, b in zip(v, JTy))
    assert lhs == pytest.approx(rhs, rel=1e-8)


def test_projection_gradient_special_cases():
    """Interior pair: identity.  Width clamped (closed or inverted pair): only the centre moves, both edges get the mean
    gradient.  Centre clamped: only the width moves, gradients are +-(gb-ga)/2.  MU below eps: no gradient."""
    lim = LIM
    one = lambda a, b: (np.array([[[a], [b]]]), np.array([[-20.0, 20.0, -30.0, 30.0]]), np.array([1.0]))
    gh = (np.array([[[3.0], [5.0]]]), np.zeros((1, 4)), np.array([7.0]))
    gl, _, gm = O.validate_adjoint(lim, *one(-10.0, 12.0), *gh)
    assert np.array_equal(gl.ravel(), [3.0, 5.0]) and gm[0] == 7.0
    gl, _, _ = O.validate_adjoint(lim, *one(4.0, 4.2), *gh)            # w = 0.2 < 0.5
    assert np.allclose(gl.ravel(), [4.0, 4.0])
    gl, _, _ = O.validate_adjoint(lim, *one(150.0, 160.0), *gh)        # c = 155 > F
    assert np.allclose(gl.ravel(), [-1.0, 1.0])
    lv, jw, _ = one(-10.0, 12.0)
    _, _, gm = O.validate_adjoint(lim, lv, jw, np.array([0.05]), *gh)
    assert gm[0] == 0.0


def masks_and_dose(seed, shape=(6, 7, 8)):
    rng = np.random.Generator(np.random.PCG64(seed))
    dose = rng.uniform(0.0, 4.0, size=shape).astype(np.float32)
    m = [rng.random(shape) < p for p in (0.2, 0.3, 0.25)]               # overlapping structures
    bits = sum((mk.astype(np.uint32) << s) for s, mk in enumerate(m))
    return dose, m, bits


@pytest.mark.parametrize("power", [1, 2])
def test_objective_matches_eq10_written_out_and_its_gradient(power):
    """Eq. 10: L = lam_PTV ||D_PTV - D_presc||_1 + sum_s lam_s ||D_s||_1 with numpy norms on the masked
    voxel vectors (power 2: the squared 2-norms); gradient against central differences of L (exact for the quadratic; for
    the 1-norm on voxels away from D = p)."""
    dose, m, bits = masks_and_dose(5)
    lam, presc = np.array([100.0, 1.0, 10.0]), np.array([3.0, 0.0, 0.0])
    L, g = O.objective(dose, bits, lam, presc, power)
    d64 = dose.astype(np.float64)
    want = sum(l * (np.linalg.norm(d64[mk] - p, 1) if power == 1 else np.linalg.norm(d64[mk] - p, 2) ** 2) for l, p, mk in zip(lam, presc, m))
    assert L == pytest.approx(want, rel=1e-12)
    rng = np.random.Generator(np.random.PCG64(55))
    for idx in zip(*[rng.integers(0, n, 12) for n in dose.shape]):
        h = 2.0 ** -8                                                   # exactly representable in float32 next to doses of O(1)
        dp, dm_ = dose.copy(), dose.copy()
        dp[idx] += h
        dm_[idx] -= h
        fd = (O.objective(dp, bits, lam, presc, power)[0] - O.objective(dm_, bits, lam, presc, power)[0]) / (float(dp[idx]) - float(dm_[idx]))
        assert g[idx] == pytest.approx(fd, rel=1e-5, abs=1e-9)
    assert not g[~(m[0] | m[1] | m[2])].any()


def test_objective_closed_forms():
    """Uniform dose d on one structure of N voxels: L1 = lam N |d - p|, L2 = lam N (d - p)^2; dose equal to the prescription:
    L = 0 and g = 0 for both powers."""
    shape = (4, 5, 6)
    bits = np.zeros(shape, np.uint32)
    bits[1:3] = 1
    N = int((bits > 0).sum())
    dose = np.full(shape, 2.5, np.float32)
    assert O.objective(dose, bits, [4.0], [3.0], 1)[0] == pytest.approx(4.0 * N * 0.5)
    assert O.objective(dose, bits, [4.0], [3.0], 2)[0] == pytest.approx(4.0 * N * 0.25)
    for power in (1, 2):
        L, g = O.objective(np.full(shape, 3.0, np.float32), bits, [4.0], [3.0], power)
        assert L == 0.0 and not g.any()


def test_jaw_tracking_equals_the_independent_numpy_routine():
    """workloads.track_jaws (the input generator, numpy) and orc_track_jaws (C) state the same recipe independently."""
    wl = W.config5()
    bounds = np.asarray(wl.model["leaf_bounds_mm"], np.float64)
    lv = wl.leaves.astype(np.float64)
    lv[3] = 0.0                                                         # a control point with every pair closed
    got = O.track_jaws(bounds, lv, 5.0, 0.6)
    want = W.track_jaws(lv, bounds, margin=5.0)
    assert np.array_equal(got, want)
    assert np.array_equal(got[3], [-5.0, 5.0, bounds[0], bounds[-1]])


def test_normalised_gradient_step_moves_by_exactly_the_step():
    rng = np.random.Generator(np.random.PCG64(8))
    lv, mu = rng.uniform(-50, 50, (5, 2, 9)), rng.uniform(1, 4, 5)
    gl, gm = rng.standard_normal(lv.shape), rng.standard_normal(mu.shape)
    nl, nm = O.plan_step(0.5, 0.05, gl, gm, lv, mu)
    assert np.abs(nl - lv).max() == pytest.approx(0.5, rel=1e-12) and np.abs(nm - mu).max() == pytest.approx(0.05, rel=1e-12)
    assert np.allclose(nl - lv, -0.5 * gl / np.abs(gl).max(), rtol=1e-12, atol=1e-15)
    assert (np.sign(nl - lv) == -np.sign(gl)).all()                    # a descent direction, entry by entry
    zl, zm = O.plan_step(0.5, 0.05, np.zeros_like(gl), gm, lv, mu)      # a zero gradient group does not move
    assert np.array_equal(zl, lv) and not np.array_equal(zm, mu)
