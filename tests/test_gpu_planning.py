"""GPU parity of the planning-loop steps against the float64 oracle, through the C ABI: the Eq. 1-3
projection and its transposed Jacobian, the objective (Eq. 10 and quadratic) with dL/dDose, jaw tracking, the normalised
gradient step, a short loop on a tiny workload run on both sides, and the c5 planning loop of BASELINE.json configs[4]
checked at iterations 1 and 20 by feeding the GPU loop's current parameters to the oracle."""
import numpy as np
import pytest

from paper_2512_18863_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def limits_pair(d):
    from oracle import oracle as O
    from paper_2512_18863_b200 import PdrtLimits
    return PdrtLimits(**d), O.plan_limits(d["leaf_w_min"], d["leaf_F"], d["jaw_w_min"], d["jaw_Fx"], d["jaw_Fy"], d["mu_eps"])


def np64(t):
    return t.double().cpu().numpy()


def test_projection_and_its_transpose(torch):
    from oracle import oracle as O
    from paper_2512_18863_b200 import Engine
    wl = W.tiny(seed=41, n_cp=9, n_pairs=13)
    eng = Engine(wl.grid, wl.model, wl.density)
    rng = np.random.Generator(np.random.PCG64(41))
    lv = rng.uniform(-60, 60, wl.leaves.shape).astype(np.float32)         # unordered pairs, centres beyond the travel range
    jw = rng.uniform(-60, 60, wl.jaws.shape).astype(np.float32)
    mu = rng.uniform(-1, 3, wl.mu.shape).astype(np.float32)
    glim, olim = limits_pair(dict(leaf_w_min=0.5, leaf_F=25.0, jaw_w_min=2.0, jaw_Fx=30.0, jaw_Fy=20.0, mu_eps=0.1))
    got = eng.validate(glim, lv, jw, mu)
    want = O.validate(olim, lv, jw, mu)
    for g, w in zip(got, want):
        assert np.abs(np64(g) - w).max() <= 1e-5
    gh = [rng.standard_normal(a.shape).astype(np.float32) for a in (lv, jw, mu)]
    got = eng.validate_backward(glim, lv, jw, mu, *gh)
    want = O.validate_adjoint(olim, lv, jw, mu, *gh)
    for g, w in zip(got, want):
        assert np.abs(np64(g) - w).max() <= 1e-6 * max(np.abs(w).max(), 1.0)
    assert eng.mu_epsilon(0.6, 2.0, 6.0) == pytest.approx(O.mu_epsilon(0.6, 2.0, 6.0), rel=1e-6)


@pytest.mark.parametrize("power", [1, 2])
def test_objective_and_dose_gradient(torch, power):
    from oracle import oracle as O
    from paper_2512_18863_b200 import Engine
    wl = W.config2()
    wl.masks = W.pelvis_masks(wl.grid)
    eng = Engine(wl.grid, wl.model, wl.density)
    bits, lam, presc = W.structure_bits(wl)
    bits[10:20, 30:60, 30:70] |= np.uint32(1 << 1) | np.uint32(1 << 2)     # overlapping structures
    rng = np.random.Generator(np.random.PCG64(50 + power))
    dose = rng.uniform(0, 4, bits.shape).astype(np.float32)
    dose[bits == 0][:10] = 0
    loss, g = eng.objective(torch.from_numpy(dose).cuda(), torch.from_numpy(bits.view(np.int32)).cuda(), lam, presc, power)
    L, gref = O.objective(dose, bits, lam, presc, power)
    assert float(loss[0]) == pytest.approx(L, rel=1e-9)
    assert np.abs(np64(g) - gref).max() <= 1e-6 * np.abs(gref).max()


def test_jaw_tracking_and_step(torch):
    from oracle import oracle as O
    from paper_2512_18863_b200 import Engine
    wl = W.tiny(seed=43, n_cp=11, n_pairs=37)                             # more pairs than lanes
    eng = Engine(wl.grid, wl.model, wl.density)
    lv = wl.leaves.copy()
    lv[4] = 0.0                                                           # no pair open: all count
    lv[5, 1] = lv[5, 0] + 0.3                                             # all below the open gap
    jaws = eng.track_jaws(lv, 5.0, 0.6)
    want = O.track_jaws(wl.model["leaf_bounds_mm"], lv, 5.0, 0.6)
    assert np.abs(np64(jaws) - want).max() <= 1e-5
    rng = np.random.Generator(np.random.PCG64(43))
    gl, gm = rng.standard_normal(lv.shape).astype(np.float32), rng.standard_normal(wl.mu.shape).astype(np.float32)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    tl, tm = t(lv), t(wl.mu)
    eng.plan_step(0.5, 0.05, t(gl), t(gm), tl, tm)
    wl_, wm_ = O.plan_step(0.5, 0.05, gl, gm, lv, wl.mu)
    assert np.abs(np64(tl) - wl_).max() <= 1e-5 and np.abs(np64(tm) - wm_).max() <= 1e-6
    tl2, tm2 = t(lv), t(wl.mu)
    eng.plan_step(0.5, 0.05, t(np.zeros_like(gl)), t(gm), tl2, tm2)       # zero gradient group: no move
    assert torch.equal(tl2, t(lv))


def oracle_iteration(orc, O, olim, wl, bits, lam, presc, leaves, mu, steps=(0.5, 0.05)):
    """One planning iteration on the oracle side (float64), the same call sequence as planning.PlanLoop.iterate."""
    n_cp = leaves.shape[0]
    pl, _, pm = O.validate(olim, leaves, np.zeros((n_cp, 4)), mu)
    jaws = O.track_jaws(wl.model["leaf_bounds_mm"], pl, 5.0, 0.6)
    dose = orc.dose(pl, jaws, wl.gantry_deg, pm)
    L, g = O.objective(dose.astype(np.float32), bits, lam, presc, 2)
    gh = orc.dose_backward(pl, jaws, wl.gantry_deg, pm, g)
    gl, _, gm = O.validate_adjoint(olim, leaves, jaws, mu, *gh)
    nl, nm = O.plan_step(steps[0], steps[1], gl, gm, leaves, mu)
    return nl, nm, L


def test_short_loop_on_both_sides(torch):
    """Four planning iterations on a small case, run independently on the GPU and on the oracle: the variables stay together."""
    from oracle import oracle as O
    from oracle.oracle import Oracle
    from paper_2512_18863_b200 import Engine
    from paper_2512_18863_b200.planning import PlanLoop
    wl = W.tiny(seed=44, n_cp=6, nx=40, ny=36, nz=18, kernel_size=7, flu=(26, 22), head_scatter=False)
    Z, Y, X = W.voxel_coords(wl.grid)
    wl.masks = {"target": ((X ** 2 + Y ** 2 + Z ** 2) <= 18.0 ** 2, 100.0, 0.05), "oar": (((X - 30) ** 2 + Y ** 2 + Z ** 2) <= 15.0 ** 2, 10.0, None)}
    bits, lam, presc = W.structure_bits(wl)
    lim = W.plan_limits(wl)
    glim, olim = limits_pair(lim)
    eng, orc = Engine(wl.grid, wl.model, wl.density), Oracle(wl.grid, wl.model, wl.density)
    loop = PlanLoop(eng, wl.leaves, wl.mu, wl.gantry_deg, glim, bits, lam, presc, power=2)
    lv, mu = wl.leaves.astype(np.float64), wl.mu.astype(np.float64)
    for it in range(4):
        loop.iterate()
        lv, mu, L = oracle_iteration(orc, O, olim, wl, bits, lam, presc, lv, mu)
        assert float(loop.loss[0]) == pytest.approx(L, rel=1e-4), f"loss at iteration {it + 1}"
    assert np.abs(np64(loop.leaves) - lv).max() <= 2e-3 and np.abs(np64(loop.mu) - mu).max() <= 2e-4


def test_config5_planning_loop_iterations_1_and_20(torch):
    """c5 (BASELINE.json configs[4]): 256x256x160 @ 2 mm, 2 x 178 control points, k = 31, 20 planning iterations on the device.
    At iterations 1 and 20 the loop's current projected parameters are fed to the oracle: sampled dose voxels, the objective
    and dL/dDose on the GPU dose, sampled gradient rows, and the update of the variables."""
    from oracle import oracle as O
    from oracle.oracle import Oracle
    from paper_2512_18863_b200 import Engine
    from paper_2512_18863_b200.planning import PlanLoop
    from test_gpu_parity import assert_grad, sample_voxels
    wl = W.config5()
    bits, lam, presc = W.structure_bits(wl)
    glim, olim = limits_pair(W.plan_limits(wl))
    eng, orc = Engine(wl.grid, wl.model, wl.density), Oracle(wl.grid, wl.model, wl.density)
    loop = PlanLoop(eng, wl.leaves, wl.mu, wl.gantry_deg, glim, bits, lam, presc, power=2)
    losses = []
    for it in range(1, 21):
        raw_l, raw_m = np64(loop.leaves), np64(loop.mu)
        loop.forward_backward()
        losses.append(float(loop.loss[0]))
        if it in (1, 20):
            pl, pm, jw = np64(loop.p_leaves), np64(loop.p_mu), np64(loop.jaws)
            wl_, _, wm_ = O.validate(olim, raw_l, np.zeros_like(jw), raw_m)
            assert np.abs(pl - wl_).max() <= 1e-4 and np.abs(pm - wm_).max() <= 1e-6, f"projection at iteration {it}"
            assert np.abs(jw - O.track_jaws(wl.model["leaf_bounds_mm"], pl, 5.0, 0.6)).max() <= 1e-4, f"jaws at iteration {it}"
            d = loop.dose.cpu().numpy()
            ijk, pick = sample_voxels(d, 90, 500 + it)
            ref = orc.dose_at(pl, jw, wl.gantry_deg, pm, ijk)
            assert np.abs(d.reshape(-1)[pick] - ref).max() <= 1e-4 * ref.max(), f"dose at iteration {it}"
            L, gref = O.objective(d, bits, lam, presc, 2)
            assert losses[-1] == pytest.approx(L, rel=1e-9)
            g = loop.g.cpu().numpy()
            assert np.abs(g - gref).max() <= 1e-6 * np.abs(gref).max()
            cps = [3, 180, 355]
            rl, rj, rm = orc.dose_backward(pl[cps], jw[cps], wl.gantry_deg[cps], pm[cps], g)
            idx = torch.as_tensor(cps, device="cuda")
            assert_grad(loop.gh[2][idx], rm, f"d_mu at iteration {it}")
            assert_grad(loop.gh[0][idx], rl, f"d_leaves at iteration {it}")
        gh = [np64(t) for t in loop.gh]
        loop.update()
        if it in (1, 20):
            gl, _, gm = O.validate_adjoint(olim, raw_l, np64(loop.jaws), raw_m, *gh)
            nl, nm = O.plan_step(0.5, 0.05, gl, gm, raw_l, raw_m)
            assert np.abs(np64(loop.leaves) - nl).max() <= 1e-4 and np.abs(np64(loop.mu) - nm).max() <= 1e-5, f"update at iteration {it}"
            assert np.abs(np64(loop.leaves) - raw_l).max() == pytest.approx(0.5, rel=1e-4)
    assert losses[-1] < losses[0], "the normalised-gradient steps reduce the objective"
