"""GPU parity of the collimator rotation (pdrt_set_collimator) against the oracle: the rotated
fluence map, the dose and the gradients, including quarter turns and the removal of the angles."""
import numpy as np
import pytest

from paper_2512_18863_b200 import workloads as W
from test_gpu_parity import assert_dose, assert_grad, pair

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


CASES = [
    dict(seed=91, nx=40, ny=36, nz=18, kernel_size=7, n_cp=4, flu=(26, 22)),
    dict(seed=92, nx=44, ny=40, nz=30, spacing=3.0, kernel_size=9, n_cp=5, flu=(30, 34), flu_d=2.5, n_pairs=9, head_scatter=False),
]
ANGLES = {91: [0.0, 17.0, -64.0, 90.0], 92: [135.0, -180.0, 3.0, 270.0, -33.0]}


@pytest.mark.parametrize("case", CASES, ids=lambda c: f"seed{c['seed']}")
def test_collimator_rotation(torch, case):
    wl = W.tiny(**case)
    coll = np.asarray(ANGLES[case["seed"]], np.float32)
    eng, orc = pair(wl)
    eng.set_collimator(coll)
    phim = eng.stage_fluence(wl.leaves, wl.jaws).double().cpu().numpy()
    for b in range(wl.n_cp):
        ref = orc.rotate_map(coll[b], orc.fluence(wl.leaves[b], wl.jaws[b]))
        assert np.abs(phim[b] - ref).max() <= 5e-6 * ref.max(), f"rotated fluence map cp {b}"
    d_ref = orc.dose_coll(wl.leaves, wl.jaws, wl.gantry_deg, coll, wl.mu)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), d_ref, "dose with collimator angles")
    g = W.seeded_dose_gradient(wl, seed=case["seed"])
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward_coll(wl.leaves, wl.jaws, wl.gantry_deg, coll, wl.mu, g)
    assert_grad(dm, rm, "coll d_mu"); assert_grad(dj, rj, "coll d_jaws"); assert_grad(dl, rl, "coll d_leaves")
    # a different number of control points than the angles were set for is an error; removing them restores the plain path
    from paper_2512_18863_b200 import PdrtError
    with pytest.raises(PdrtError):
        eng.dose(wl.leaves[:2], wl.jaws[:2], wl.gantry_deg[:2], wl.mu[:2])
    eng.set_collimator(None)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "angles removed")


def test_collimator_on_c2_fields(torch):
    """c2's irregular 110 x 250 mm apertures turned by 30-90 degrees: the rotated support leaves the map on two sides."""
    wl = W.config2()
    coll = np.asarray([30.0, 45.0, 60.0, 90.0, -75.0], np.float32)
    eng, orc = pair(wl)
    eng.set_collimator(coll)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose_coll(wl.leaves, wl.jaws, wl.gantry_deg, coll, wl.mu), "c2 with collimator")
    g = W.seeded_dose_gradient(wl, seed=93)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward_coll(wl.leaves, wl.jaws, wl.gantry_deg, coll, wl.mu, g)
    assert_grad(dm, rm, "c2 coll d_mu"); assert_grad(dj, rj, "c2 coll d_jaws"); assert_grad(dl, rl, "c2 coll d_leaves")
