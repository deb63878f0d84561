"""Pins of the divergent radiological-depth mode of the oracle (reading G24 of DESIGN.md): one
diverging ray per fluence-map pixel, depth counted per unit axial distance, depth factor T(z_ray)/T(z_cax) on the projected
fluence.  Checked against the central-axis routine, the reduction to the paper's mode in laterally homogeneous media,
closed forms under a tilted surface, the adjoint identity and finite differences."""
import numpy as np
import pytest

from oracle.oracle import Oracle
from paper_2512_18863_b200 import workloads as W


def slab_case(flu=(21, 17), gantry=0.0):
    """Slabs normal to y (the beam axis at gantry 0), odd fluence map so that one pixel sits on the axis."""
    wl = W.tiny(seed=61, nx=30, ny=34, nz=14, spacing=4.0, n_cp=2, kernel_size=5, flu=flu, head_scatter=False, gantry=[gantry, gantry])
    Z, Y, X = W.voxel_coords(wl.grid)
    depth = Y - (wl.grid["oy"] - 0.5 * wl.grid["sy"])
    rho = np.ones_like(depth)
    rho[(depth >= 24) & (depth < 48)] = 0.3
    rho[(depth >= 80) & (depth < 96)] = 1.7
    wl.density = rho.astype(np.float32)
    wl.grid["iso"] = (0.0, 0.0, 0.0)
    return wl


def test_axis_ray_equals_the_central_axis_routine():
    wl = W.tiny(seed=62, flu=(21, 17), gantry=[33.0, 211.0, 90.0])       # random density, oblique angles
    orc = Oracle(wl.grid, wl.model, wl.density)
    for ga in wl.gantry_deg:
        zf = orc.fan_depth(ga)
        assert np.array_equal(zf[:, 8, 10], orc.radiological_depth(ga))  # pixel (a,b) = (10,8): uf = vf = 0


def test_reduces_to_the_papers_mode_in_laterally_homogeneous_slabs():
    """Slabs normal to the axis: every ray reproduces the central-axis depth profile (depth per unit axial distance), the
    factor is identically 1 and the dose equals the paper-mode dose."""
    wl = slab_case()
    orc = Oracle(wl.grid, wl.model, wl.density)
    zc = orc.radiological_depth(0.0)
    zf = orc.fan_depth(0.0)
    inside = np.abs(zf - zc[:, None, None]) <= 1e-9 * max(zc.max(), 1.0)
    # rays that leave the grid box sideways stop accumulating: compare the rays that stay inside (the central 11 x 9 pixels)
    assert inside[:, 4:13, 5:16].all()
    F = orc.fan_factor(zf, zc)
    assert np.abs(F[:, 4:13, 5:16] - 1.0).max() <= 1e-9
    jaws = np.tile([-10.0, 10.0, -8.0, 8.0], (2, 1))                      # a field well inside those rays
    d0 = orc.dose(wl.leaves, jaws, wl.gantry_deg, wl.mu)
    d1 = orc.dose_fan(wl.leaves, jaws, wl.gantry_deg, wl.mu)
    assert d0.max() > 0 and np.abs(d1 - d0).max() <= 1e-9 * d0.max()


def test_tilted_surface_closed_form():
    """Water below the tilted plane y = y0 + alpha x, gantry 0 (source at y = -SID, axis along +y): ray (a,b) enters at
    t_e = (y0 - src_y) / (1 - alpha uf/SID) and z_fan(k) = max(0, d_k - t_e) up to the voxelisation of the surface."""
    wl = W.tiny(seed=63, nx=44, ny=40, nz=12, spacing=3.0, n_cp=1, kernel_size=5, flu=(25, 9), flu_d=3.0, head_scatter=False, gantry=[0.0])
    wl.grid["iso"] = (0.0, 0.0, 0.0)
    Z, Y, X = W.voxel_coords(wl.grid)
    alpha, y0 = 0.5, -20.0
    wl.density = (Y > y0 + alpha * X).astype(np.float32)
    orc = Oracle(wl.grid, wl.model, wl.density)
    zf = orc.fan_depth(0.0)
    sid = wl.model["sid_mm"]
    uf = (np.arange(25) - 12) * 3.0
    d = sid + orc.m["beam_wmin"] + np.arange(orc.m["beam_nw"]) * orc.m["beam_dw"]
    t_e = (y0 + sid) / (1.0 - alpha * uf / sid)                           # src_x = 0, src_y = -SID
    want = np.maximum(0.0, d[:, None] - t_e[None, :])
    got = zf[:, 4, :]                                                     # the row vf = 0
    ok = (np.abs(uf) <= 30)[None, :] & (d[:, None] < sid + 50)            # rays and depths that stay inside the grid
    assert np.abs(got - want)[np.broadcast_to(ok, got.shape)].max() <= 3.0   # one voxel of surface smearing
    # the sign of the tilt matters: rays at +u enter later (deeper surface) than rays at -u by about alpha * 2 u
    assert (got[20, 22] - got[20, 2]) < -0.8 * alpha * 60.0


def test_depth_term_is_the_plane_integral_of_the_kernel():
    """T(z) = 2 pi (A/a + B/b) = the integral of (A e^{-ar} + B e^{-br})/r over the plane; with the synthetic model's
    A = P a / 2 pi, B = S b / 2 pi (workloads.common_model) that is P(z) + S(z) at the table nodes, linear in between."""
    wl = W.tiny(seed=64)
    orc = Oracle(wl.grid, wl.model, wl.density)
    z = np.arange(256) * 2.0
    P = (1.0 - np.exp(-0.25 * z)) * np.exp(-0.004 * z)
    S = 0.35 * (1.0 - np.exp(-0.01 * z)) * np.exp(-0.004 * z)
    for n in (0, 1, 7, 100, 255):
        assert orc.depth_term(z[n]) == pytest.approx(P[n] + S[n], rel=2e-6, abs=1e-12)      # tables are float32 inputs
    assert orc.depth_term(15.0) == pytest.approx(0.5 * (P[7] + S[7] + P[8] + S[8]), rel=2e-6)
    assert orc.depth_term(-3.0) == pytest.approx(0.0, abs=1e-12) and orc.depth_term(1e4) == pytest.approx(P[255] + S[255], rel=2e-6)
    # radial quadrature of K over the plane at one node
    m = orc.m
    A, a, B, b = (float(m[k][50]) for k in ("kA", "ka", "kB", "kb"))
    r = (np.arange(400000) + 0.5) * 0.005
    quad = np.sum((A * np.exp(-a * r) + B * np.exp(-b * r)) / r * 2 * np.pi * r) * 0.005
    assert orc.depth_term(100.0) == pytest.approx(quad, rel=1e-4)


def test_factor_is_one_where_the_axis_term_vanishes_and_a_ratio_elsewhere():
    wl = W.tiny(seed=65, flu=(9, 7))
    orc = Oracle(wl.grid, wl.model, wl.density)
    zf = np.random.Generator(np.random.PCG64(65)).uniform(0, 200, orc.fan_shape)
    zc = np.linspace(0.0, 150.0, orc.fan_shape[0])
    zc[:3] = 0.0                                                          # slices in front of the surface: T = 0
    F = orc.fan_factor(zf, zc)
    assert np.array_equal(F[:3], np.ones_like(F[:3]))
    assert F[10, 3, 4] == pytest.approx(orc.depth_term(zf[10, 3, 4]) / orc.depth_term(zc[10]), rel=1e-13)


def test_weighted_projection_adjoint_identity_and_interpolation():
    wl = W.tiny(seed=66, flu=(14, 12))
    orc = Oracle(wl.grid, wl.model, wl.density)
    rng = np.random.Generator(np.random.PCG64(66))
    F = rng.uniform(0.5, 1.5, orc.fan_shape)
    x, y = rng.standard_normal(orc.flu_shape), rng.standard_normal(orc.beam_shape)
    Ax = orc.apply_fan_factor(F, orc.project(x))
    ATy = orc.project_adjoint(orc.apply_fan_factor(F, y))
    assert float((Ax * y).sum()) == pytest.approx(float((x * ATy).sum()), rel=1e-12)
    # a factor that is constant per slice scales the slice; a factor linear in the pixel index is reproduced exactly inside the map
    Fc = np.broadcast_to(np.linspace(0.7, 1.3, orc.fan_shape[0])[:, None, None], orc.fan_shape).copy()
    v = rng.uniform(1, 2, orc.beam_shape)
    assert np.allclose(orc.apply_fan_factor(Fc, v), v * Fc[:, :1, :1], rtol=1e-13)
    a = np.arange(orc.fan_shape[2])
    Fl = np.broadcast_to(1.0 + 0.01 * a[None, None, :], orc.fan_shape).copy()
    k = orc.fan_shape[0] // 2
    mag = orc.m["sid"] / (orc.m["sid"] + orc.m["beam_wmin"] + k * orc.m["beam_dw"])
    i = np.arange(orc.m["beam_nu"])
    fa = mag * (i - 0.5 * (orc.m["beam_nu"] - 1)) * orc.m["beam_du"] / orc.m["flu_du"] + 0.5 * (orc.m["flu_nu"] - 1)
    want = 1.0 + 0.01 * np.clip(fa, 0, orc.fan_shape[2] - 1)
    got = orc.apply_fan_factor(Fl, np.ones(orc.beam_shape))[k, 0, :]
    assert np.allclose(got, want, rtol=1e-12)


def test_gradients_of_the_fan_mode_vs_finite_differences():
    wl = W.tiny(seed=67, n_cp=2, nx=22, ny=20, nz=10, kernel_size=5, flu=(16, 12), head_scatter=False)
    orc = Oracle(wl.grid, wl.model, wl.density)
    rng = np.random.Generator(np.random.PCG64(67))
    g = rng.standard_normal(orc.dose_shape).astype(np.float32)
    lv, jw, mu = wl.leaves.astype(np.float64), wl.jaws.astype(np.float64), wl.mu.astype(np.float64)
    dl, dj, dm = orc.dose_backward_fan(lv, jw, wl.gantry_deg, mu, g)
    L = lambda l, j, m: float((orc.dose_fan(l, j, wl.gantry_deg, m) * g).sum())
    h = 1e-4
    for (b, bank, i) in ((0, 0, 2), (1, 1, 3), (0, 1, 4)):
        p, q = lv.copy(), lv.copy()
        p[b, bank, i] += h; q[b, bank, i] -= h
        assert dl[b, bank, i] == pytest.approx((L(p, jw, mu) - L(q, jw, mu)) / (2 * h), rel=1e-6, abs=1e-10)
    for (b, e) in ((0, 0), (1, 3)):
        p, q = jw.copy(), jw.copy()
        p[b, e] += h; q[b, e] -= h
        assert dj[b, e] == pytest.approx((L(lv, p, mu) - L(lv, q, mu)) / (2 * h), rel=1e-6, abs=1e-10)
    p, q = mu.copy(), mu.copy()
    p[1] += h; q[1] -= h
    assert dm[1] == pytest.approx((L(lv, jw, p) - L(lv, jw, q)) / (2 * h), rel=1e-8)
    # and the mode differs from the paper's on this laterally inhomogeneous phantom
    assert np.abs(orc.dose_fan(lv, jw, wl.gantry_deg, mu) - orc.dose(lv, jw, wl.gantry_deg, mu)).max() > 1e-3 * orc.dose(lv, jw, wl.gantry_deg, mu).max()


def test_fan_mode_with_collimator_rotation_reduces_to_each_mode_and_matches_finite_differences():
    """orc_dose_fan_coll composes the two optional steps (rotation, then projection, then the depth factor).  Pins: collimator 0
    gives the fan-mode dose bit for bit; in slabs normal to the axis (factor 1 on the rays that stay inside) it gives the
    collimator-mode dose; it differs from both where both steps act; its gradients match central differences of its own dose."""
    wl = W.tiny(seed=68, n_cp=2, nx=22, ny=20, nz=10, kernel_size=5, flu=(16, 12), head_scatter=False)
    orc = Oracle(wl.grid, wl.model, wl.density)
    lv, jw, mu = wl.leaves.astype(np.float64), wl.jaws.astype(np.float64), wl.mu.astype(np.float64)
    zero, coll = np.zeros(2), np.asarray([27.0, -64.0])
    assert np.array_equal(orc.dose_fan_coll(lv, jw, wl.gantry_deg, zero, mu), orc.dose_fan(lv, jw, wl.gantry_deg, mu))
    d_fc = orc.dose_fan_coll(lv, jw, wl.gantry_deg, coll, mu)
    d_f, d_c = orc.dose_fan(lv, jw, wl.gantry_deg, mu), orc.dose_coll(lv, jw, wl.gantry_deg, coll, mu)
    assert np.abs(d_fc - d_f).max() > 1e-3 * d_f.max() and np.abs(d_fc - d_c).max() > 1e-3 * d_c.max()
    # slabs normal to the axis, field well inside the rays that stay in the grid: the factor is 1, only the rotation acts
    ws = slab_case()
    os_ = Oracle(ws.grid, ws.model, ws.density)
    jaws = np.tile([-9.0, 9.0, -7.0, 7.0], (2, 1))
    c2 = np.asarray([15.0, -40.0])
    a, b = os_.dose_fan_coll(ws.leaves, jaws, ws.gantry_deg, c2, ws.mu), os_.dose_coll(ws.leaves, jaws, ws.gantry_deg, c2, ws.mu)
    assert b.max() > 0 and np.abs(a - b).max() <= 1e-9 * b.max()
    # gradients vs central differences
    rng = np.random.Generator(np.random.PCG64(68))
    g = rng.standard_normal(orc.dose_shape).astype(np.float32)
    dl, dj, dm = orc.dose_backward_fan_coll(lv, jw, wl.gantry_deg, coll, mu, g)
    L = lambda l, j, m: float((orc.dose_fan_coll(l, j, wl.gantry_deg, coll, m) * g).sum())
    h = 1e-4
    for (bb, bank, i) in ((0, 0, 2), (1, 1, 3)):
        p, q = lv.copy(), lv.copy()
        p[bb, bank, i] += h; q[bb, bank, i] -= h
        assert dl[bb, bank, i] == pytest.approx((L(p, jw, mu) - L(q, jw, mu)) / (2 * h), rel=1e-6, abs=1e-10)
    p, q = jw.copy(), jw.copy()
    p[1, 2] += h; q[1, 2] -= h
    assert dj[1, 2] == pytest.approx((L(lv, p, mu) - L(lv, q, mu)) / (2 * h), rel=1e-6, abs=1e-10)
    p, q = mu.copy(), mu.copy()
    p[0] += h; q[0] -= h
    assert dm[0] == pytest.approx((L(lv, jw, p) - L(lv, jw, q)) / (2 * h), rel=1e-8)
