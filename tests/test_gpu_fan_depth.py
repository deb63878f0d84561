"""GPU parity of the divergent radiological-depth mode (PDRT_DEPTH_FAN) against the oracle's fan
functions: the depth factor at the ray nodes, the dose and the gradients; and the reduction to the paper's mode."""
import numpy as np
import pytest

from paper_2512_18863_b200 import workloads as W
from test_gpu_parity import assert_dose, assert_grad, fluence_support_mask

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def pair(wl):
    from oracle.oracle import Oracle
    from paper_2512_18863_b200 import Engine
    eng = Engine(wl.grid, dict(wl.model, depth_mode=1), wl.density)
    return eng, Oracle(wl.grid, wl.model, wl.density)


CASES = [
    dict(seed=71, nx=40, ny=36, nz=16, kernel_size=7, n_cp=3, flu=(26, 22)),
    dict(seed=72, nx=37, ny=45, nz=21, spacing=3.0, kernel_size=9, n_cp=4, flu=(30, 26), flu_d=2.5, head_scatter=False),
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: f"seed{c['seed']}")
def test_fan_factor_dose_and_gradients(torch, case):
    wl = W.tiny(**case)
    eng, orc = pair(wl)
    F = eng.stage_fan_factor(wl.leaves, wl.jaws, wl.gantry_deg).double().cpu().numpy()
    for b in range(wl.n_cp):
        ref = orc.fan_factor(orc.fan_depth(wl.gantry_deg[b]), orc.radiological_depth(wl.gantry_deg[b]))
        box = fluence_support_mask(wl, b, extra=1)                 # the rays traced: support bbox grown by one pixel
        rows, cols = np.flatnonzero(box.any(axis=1)), np.flatnonzero(box.any(axis=0))
        sl = (slice(None), slice(rows[0], rows[-1] + 1), slice(cols[0], cols[-1] + 1))
        assert np.abs(F[b][sl] - ref[sl]).max() <= 2e-5 * np.abs(ref[sl]).max(), f"depth factor cp {b}"
    d_ref = orc.dose_fan(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), d_ref, "fan dose")
    assert np.abs(d_ref - orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)).max() > 1e-3 * d_ref.max()      # the mode matters here
    g = W.seeded_dose_gradient(wl, seed=case["seed"])
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward_fan(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dm, rm, "fan d_mu"); assert_grad(dj, rj, "fan d_jaws"); assert_grad(dl, rl, "fan d_leaves")
    eng.set_depth_mode(0)                                          # back to the paper's mode on the same engine
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "axis dose")


def test_fan_mode_on_the_slab_phantom_equals_the_papers_mode(torch):
    """c2's slabs are normal to y; at gantry 0 and 180 every diverging ray sees the central-axis profile: the factor is 1
    where the rays stay inside the grid and the dose equals the axis-mode dose; at the oblique angles it differs."""
    wl = W.config2()
    wl.gantry_deg = np.asarray([0.0, 180.0, 0.0, 180.0, 0.0], np.float32)
    wl.jaws[:] = (-40.0, 40.0, -60.0, 60.0)
    eng, orc = pair(wl)
    d_fan = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    eng.set_depth_mode(0)
    d_axis = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert float((d_fan - d_axis).abs().max()) <= 2e-5 * float(d_axis.max())
    assert_dose(d_fan, orc.dose_fan(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "c2 fan dose")


def test_fan_mode_on_the_pelvis_phantom_sampled(torch):
    """c3-sized case (curved body surface, bones, air pocket): 12 control points of the arc, whole grid."""
    wl = W.config3()
    idx = np.arange(0, 178, 15)
    wl.leaves, wl.jaws, wl.gantry_deg, wl.mu = wl.leaves[idx], wl.jaws[idx], wl.gantry_deg[idx], wl.mu[idx]
    eng, orc = pair(wl)
    d = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    ref = orc.dose_fan(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert_dose(d, ref, "pelvis fan dose")
    assert np.abs(ref - orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)).max() > 1e-3 * ref.max()


def test_fan_mode_with_collimator_rotation(torch):
    """Both optional steps at once (pdrt_set_collimator on a PDRT_DEPTH_FAN engine) against the oracle's composition."""
    wl = W.tiny(seed=73, nx=40, ny=36, nz=16, kernel_size=7, n_cp=3, flu=(26, 22))
    eng, orc = pair(wl)
    coll = np.asarray([25.0, -70.0, 130.0], np.float32)
    eng.set_collimator(coll)
    d_ref = orc.dose_fan_coll(wl.leaves, wl.jaws, wl.gantry_deg, coll, wl.mu)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), d_ref, "fan + collimator dose")
    assert np.abs(d_ref - orc.dose_fan(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)).max() > 1e-3 * d_ref.max()
    g = W.seeded_dose_gradient(wl, seed=73)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward_fan_coll(wl.leaves, wl.jaws, wl.gantry_deg, coll, wl.mu, g)
    assert_grad(dm, rm, "fan + collimator d_mu"); assert_grad(dj, rj, "fan + collimator d_jaws"); assert_grad(dl, rl, "fan + collimator d_leaves")
