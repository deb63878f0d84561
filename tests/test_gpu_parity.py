"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element, on the same
seeded inputs.  Acceptance (BASELINE.json north_star): dose  max|D_gpu - D_orc| <= 1e-4 * max(D_orc);
gradients  ||g_gpu - g_orc||_2 / ||g_orc||_2 <= 1e-3 per group (leaves, jaws, MU) and max-abs <= 1e-3 * max|g_orc|.
"""
import numpy as np
import pytest

from paper_2512_18863_b200 import workloads as W

pytestmark = pytest.mark.gpu

DOSE_TOL = 1e-4
GRAD_TOL = 1e-3


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def pair(wl):
    from oracle.oracle import Oracle
    from paper_2512_18863_b200 import Engine
    return Engine(wl.grid, wl.model, wl.density), Oracle(wl.grid, wl.model, wl.density)


def assert_dose(gpu, orc, what=""):
    gpu = gpu.double().cpu().numpy() if hasattr(gpu, "cpu") else np.asarray(gpu, np.float64)
    scale = np.abs(orc).max()
    err = np.abs(gpu - orc).max()
    assert np.isfinite(gpu).all(), what
    assert scale > 0, f"{what}: oracle dose is identically zero"
    assert err <= DOSE_TOL * scale, f"{what}: max err {err:.3e} vs {DOSE_TOL}*max {scale:.3e} (ratio {err / scale:.2e})"
    return err / scale


def assert_grad(gpu, orc, what=""):
    gpu = gpu.double().cpu().numpy()
    assert np.isfinite(gpu).all(), what
    n = np.linalg.norm(orc)
    assert n > 0, f"{what}: oracle gradient is identically zero"
    rel = np.linalg.norm(gpu - orc) / n
    mx = np.abs(gpu - orc).max() / np.abs(orc).max()
    assert rel <= GRAD_TOL and mx <= GRAD_TOL, f"{what}: rel L2 {rel:.2e}, max-abs ratio {mx:.2e}"
    return rel


def fluence_support_mask(wl, b, extra=0):
    """Pixels whose Phi0 can be non-zero (pixels overlapped by the jaw opening), dilated by the largest Gaussian half-widths
    ceil(3 sigma / D) of the penumbra and head-scatter blurs (G13): where dL/dPhimap is consumed."""
    m = wl.model
    nu, nv, du, dv = m["flu_nu"], m["flu_nv"], m["flu_du"], m["flu_dv"]
    x1, x2, y1, y2 = (float(v) for v in wl.jaws[b])
    eu = (np.arange(nu + 1) - 0.5 * nu) * du
    ev = (np.arange(nv + 1) - 0.5 * nv) * dv
    ua = (np.minimum(eu[1:], x2) - np.maximum(eu[:-1], x1)) > 0
    vb = (np.minimum(ev[1:], y2) - np.maximum(ev[:-1], y1)) > 0
    sig = [m["fwhm_mlc_mm"] / 2.354820045, m["fwhm_jaw_mm"] / 2.354820045] + [float(x) for x in np.asarray(m["hs_sigma_mm"])[:m["n_hs"]]]
    tu = max(int(np.ceil(3.0 * sg / du)) for sg in [sig[0]] + sig[2:])
    tv = max(int(np.ceil(3.0 * sg / dv)) for sg in [sig[1]] + sig[2:])
    grow = lambda a, t: np.convolve(a.astype(int), np.ones(2 * t + 1, int))[t:t + len(a)] > 0      # dilation by t pixels
    return np.outer(grow(vb, tv + extra), grow(ua, tu + extra))


TINY_CASES = [
    dict(seed=7),
    dict(seed=8, kernel_size=3, head_scatter=False),
    dict(seed=9, kernel_size=7, nx=37, ny=29, nz=17, n_cp=4, flu=(26, 22)),
    dict(seed=10, kernel_size=11, nx=45, ny=40, nz=21, spacing=3.0, flu=(40, 30), flu_d=2.0, n_pairs=11),
    dict(seed=11, kernel_size=13, nx=70, ny=33, nz=40, spacing=2.5, flu=(48, 44), flu_d=2.5, n_pairs=9, n_cp=2),
]


@pytest.mark.parametrize("case", TINY_CASES, ids=lambda c: f"seed{c['seed']}")
def test_stages_tiny(torch, case):
    wl = W.tiny(**case)
    eng, orc = pair(wl)
    phim = eng.stage_fluence(wl.leaves, wl.jaws).double().cpu().numpy()
    zr = eng.stage_depth(wl.gantry_deg).double().cpu().numpy()
    for b in range(wl.n_cp):
        ref = orc.fluence(wl.leaves[b], wl.jaws[b])
        assert np.abs(phim[b] - ref).max() <= 2e-6 * max(ref.max(), 1e-30), f"fluence map cp {b}"
        zref = orc.radiological_depth(wl.gantry_deg[b])
        assert np.abs(zr[b] - zref).max() <= 1e-5 * max(zref.max(), 1.0), f"radiological depth cp {b}"
        db = eng.stage_beam_dose(wl.leaves[b:b + 1], wl.jaws[b:b + 1], wl.gantry_deg[b:b + 1])
        assert_dose(db, orc.beam_dose(wl.leaves[b], wl.jaws[b], wl.gantry_deg[b]), f"beam dose cp {b}")


@pytest.mark.parametrize("case", TINY_CASES, ids=lambda c: f"seed{c['seed']}")
def test_forward_backward_tiny(torch, case):
    wl = W.tiny(**case)
    eng, orc = pair(wl)
    d_ref = orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), d_ref, "dose")
    g = W.seeded_dose_gradient(wl, seed=case["seed"])
    gphi = eng.stage_grad_fluence(wl.leaves, wl.jaws, wl.gantry_deg, g).double().cpu().numpy()
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    Wt = orc.kernel_table()
    for b in range(wl.n_cp):        # dL/dPhimap on the fluence support of each control point (mask built here, not from the GPU)
        z = orc.radiological_depth(wl.gantry_deg[b])
        ref = orc.project_adjoint(orc.convolve(Wt, z, orc.resample_adjoint(wl.gantry_deg[b], g), transpose=True))
        sup = fluence_support_mask(wl, b)
        assert sup.any() and np.count_nonzero(gphi[b][sup]) > 0.9 * sup.sum(), f"dL/dPhimap cp {b}: support not covered"
        assert np.abs(gphi[b][sup] - ref[sup]).max() <= 1e-4 * np.abs(ref).max(), f"dL/dPhimap cp {b}"
        assert not gphi[b][~fluence_support_mask(wl, b, extra=1)].any(), f"dL/dPhimap cp {b}: non-zero outside the support"
    assert_grad(dm, rm, "d_mu")
    assert_grad(dj, rj, "d_jaws")
    assert_grad(dl, rl, "d_leaves")


def test_config1_water_phantom(torch):
    """c1: 64^3 water, one open 10x10 field, beam grid == patient grid (S6 is the identity)."""
    wl = W.config1()
    eng, orc = pair(wl)
    d_ref = orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    d = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert_dose(d, d_ref, "c1 dose")
    # properties on the GPU result itself: mirror symmetry of the symmetric field (P3), MU linearity (P1)
    dn = d.cpu().numpy()
    assert np.allclose(dn, dn[:, :, ::-1], rtol=1e-4, atol=1e-6 * dn.max())
    assert np.allclose(dn, dn[::-1], rtol=1e-4, atol=1e-6 * dn.max())
    d2 = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, 2.0 * wl.mu).cpu().numpy()
    assert np.allclose(d2, 2.0 * dn, rtol=1e-6)
    closed = wl.jaws.copy()
    closed[:, 1] = closed[:, 0] - 1.0
    assert float(eng.dose(wl.leaves, closed, wl.gantry_deg, wl.mu).abs().max()) == 0.0     # P2


def test_config2_slab_phantom_forward_and_backward(torch):
    """c2: heterogeneous slabs, 5 beams with irregular apertures, k = 21; forward and (beyond BASELINE) backward."""
    wl = W.config2()
    eng, orc = pair(wl)
    d_ref = orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), d_ref, "c2 dose")
    g = W.seeded_dose_gradient(wl, seed=2)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dm, rm, "c2 d_mu")
    assert_grad(dj, rj, "c2 d_jaws")
    assert_grad(dl, rl, "c2 d_leaves")


def test_edge_cases(torch):
    """Closed and inverted jaws, closed leaves, fields cut by the map / grid edge, a single control point,
    kernel sizes that run on a larger compiled variant."""
    wl = W.tiny(seed=12, n_cp=5, kernel_size=9, nx=40, ny=36, nz=14, flu=(24, 20))
    half_u = 0.5 * wl.model["flu_nu"] * wl.model["flu_du"]
    wl.jaws[0, :2] = (3.0, 3.0)                    # closed
    wl.jaws[1, :2] = (9.0, -9.0)                   # inverted
    wl.leaves[2] = 0.0                             # all pairs closed: transmission only
    wl.jaws[3] = (-10 * half_u, 10 * half_u, -1e3, 1e3)   # wider than the map and the grid
    wl.leaves[3, 0], wl.leaves[3, 1] = -1e3, 1e3
    eng, orc = pair(wl)
    d_ref = orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), d_ref, "edge dose")
    g = W.seeded_dose_gradient(wl, seed=12)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert float(dm[0]) == 0.0 and float(dm[1]) == 0.0 and float(dl[0].abs().max()) == 0.0
    assert_grad(dm, rm, "edge d_mu")
    assert_grad(dl[2:], rl[2:], "edge d_leaves")
    assert_grad(dj[2:], rj[2:], "edge d_jaws")
    for b in range(wl.n_cp):                        # single control points, one at a time
        one = eng.dose(wl.leaves[b:b + 1], wl.jaws[b:b + 1], wl.gantry_deg[b:b + 1], wl.mu[b:b + 1])
        ref = orc.dose(wl.leaves[b:b + 1], wl.jaws[b:b + 1], wl.gantry_deg[b:b + 1], wl.mu[b:b + 1])
        if ref.max() > 0:
            assert_dose(one, ref, f"edge single cp {b}")
        else:
            assert float(one.abs().max()) == 0.0


@pytest.mark.parametrize("k", [3, 5, 9, 17, 23, 33, 41, 43, 51, 55, 63, 75, 93, 125])
def test_kernel_size_sweep_small(torch, k):
    """pdrt_set_kernel_size, including sizes that have no compiled variant of their own, and sizes above 75, which run as
    NB x NB passes of shifted sub-kernels (93: 3 x 3; 125: 5 x 5)."""
    big = k > 33                       # a grid that holds the halo of the large kernels
    wl = W.tiny(seed=13, n_cp=2, kernel_size=5, nx=80 if big else 48, ny=44, nz=76 if big else 36, spacing=3.0, flu=(30, 30))
    eng, orc = pair(wl)
    eng.set_kernel_size(k)
    orc.set_kernel_size(k)
    passes = int(round(eng.info.kernel_passes ** 0.5))
    assert eng.info.kernel_size == k and passes * eng.info.kernel_size_compiled >= k and (passes == 1) == (k <= 75)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), f"k={k}")
    g = W.seeded_dose_gradient(wl, seed=k)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dm, rm, f"k={k} d_mu")
    assert_grad(dl, rl, f"k={k} d_leaves")


def test_host_entry_points_and_errors(torch):
    from paper_2512_18863_b200 import Engine, PdrtError
    wl = W.tiny(seed=14)
    eng, orc = pair(wl)
    out = torch.empty(eng.dose_shape, dtype=torch.float32).pin_memory()
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    eng.dose_host(t(wl.leaves), t(wl.jaws), t(wl.gantry_deg), t(wl.mu), out)
    assert_dose(out, orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "dose_host")
    g = W.seeded_dose_gradient(wl, seed=14)
    dl, dj, dm = (torch.empty(wl.leaves.shape).pin_memory(), torch.empty(wl.jaws.shape).pin_memory(), torch.empty(wl.mu.shape).pin_memory())
    # asynchronous download of the dose overlapping the backward call, twice in a row (the staging buffers are reused)
    hl, hj, hg, hm, hgd = t(wl.leaves), t(wl.jaws), t(wl.gantry_deg), t(wl.mu), t(g)      # stay alive until host_wait
    for rep in range(2):
        out.zero_()
        hm2 = t(wl.mu * (1 + rep))
        eng.dose_host_async(hl, hj, hg, hm2, out)
        eng.dose_backward_host(hl, hj, hg, hm, hgd, dl, dj, dm)
        eng.host_wait()
        assert_dose(out, (1 + rep) * orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), f"dose_host_async {rep}")
    eng.dose_backward_host(t(wl.leaves), t(wl.jaws), t(wl.gantry_deg), t(wl.mu), t(g), dl, dj, dm)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dl, rl, "host d_leaves"); assert_grad(dj, rj, "host d_jaws"); assert_grad(dm, rm, "host d_mu")
    w = eng.get_work()
    assert w.n_cp == wl.n_cp and w.support_voxels > 0 and w.footprint_voxels >= w.support_voxels and w.conv_macs > 0
    bad = dict(wl.model, kernel_size=8)
    with pytest.raises(PdrtError):
        Engine(wl.grid, bad, wl.density)
    with pytest.raises(PdrtError):
        eng.set_kernel_size(257)
    with pytest.raises(PdrtError):
        Engine(wl.grid, dict(wl.model, leaf_bounds_mm=np.zeros(wl.model["n_pairs"] + 1, np.float32)), wl.density)


# ---------------------------------------------------------------------------------------------------------------
# Full-size configurations, in the launch configuration bench.py times.  c3 and c4 (k = 21) are compared over the WHOLE
# dose grid and over ALL gradient rows (the oracle needs about a minute per arc on the GPU box's host cores); the other
# kernel sizes of the c4 sweep and c5 are compared on sampled voxels that the oracle computes one by one (orc_dose_at: the
# same definitions evaluated per output) and on sampled control points (gradient rows of different control points are
# independent given dL/dDose).
def sample_voxels(dose, n, seed):
    """Seeded sample of voxel indices (x, y, z): the maximum, voxels above 5 % of it, and voxels anywhere."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nz, ny, nx = dose.shape
    flat = dose.reshape(-1)
    top = int(np.argmax(flat))
    hot = np.flatnonzero(flat > 0.05 * flat[top])
    pick = np.concatenate([[top], rng.choice(hot, size=min(len(hot), (2 * n) // 3), replace=False),
                           rng.integers(0, flat.size, size=n // 3)])
    z, rem = np.divmod(pick, ny * nx)
    y, x = np.divmod(rem, nx)
    return np.stack([x, y, z], axis=1).astype(np.int32), pick


def check_sampled_dose(eng, orc, wl, n_pts, seed, what, params=None):
    lv, jw, ga, mu = params if params is not None else (wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    d = eng.dose(lv, jw, ga, mu).cpu().numpy()
    assert np.isfinite(d).all()
    ijk, pick = sample_voxels(d, n_pts, seed)
    ref = orc.dose_at(lv, jw, ga, mu, ijk)
    scale = ref.max()                                   # includes the voxel where the GPU dose peaks
    assert scale > 0
    err = np.abs(d.reshape(-1)[pick].astype(np.float64) - ref).max()
    assert err <= DOSE_TOL * scale, f"{what}: sampled max err {err:.3e} vs {DOSE_TOL}*{scale:.3e} (ratio {err / scale:.2e})"
    return d


def check_sampled_gradients(eng, orc, wl, g, cps, what, params=None):
    lv, jw, ga, mu = params if params is not None else (wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    dl, dj, dm = eng.dose_backward(lv, jw, ga, mu, g)
    rl, rj, rm = orc.dose_backward(lv[cps], jw[cps], ga[cps], mu[cps], g)
    assert np.isfinite(dl.cpu().numpy()).all() and np.isfinite(dj.cpu().numpy()).all() and np.isfinite(dm.cpu().numpy()).all()
    idx = torch_index(dl, cps)
    assert_grad(dm[idx], rm, f"{what} d_mu")
    assert_grad(dl[idx], rl, f"{what} d_leaves")
    assert_grad(dj[idx], rj, f"{what} d_jaws")


def torch_index(t, cps):
    import torch as _t
    return _t.as_tensor(np.asarray(cps), device=t.device, dtype=_t.long)


def test_config3_full_arc_forward_whole_grid(torch):
    """c3: 200x200x120 pelvis phantom, 178 control points, 60 leaf pairs, k = 21, forward — every voxel of the dose grid
    (reaches the second GATHER pass of the resampler and the long control-point lists that sampling only touched)."""
    wl = W.config3()
    eng, orc = pair(wl)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "c3 whole grid")


def test_config4_full_arc_whole_grid_and_all_gradient_rows(torch):
    """c4 at k = 21 (the configuration bench.py times): every voxel of the dose grid and all 178 gradient rows."""
    wl = W.config4(21)
    eng, orc = pair(wl)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "c4 whole grid")
    g = W.seeded_dose_gradient(wl, seed=4)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dm, rm, "c4 d_mu"); assert_grad(dj, rj, "c4 d_jaws"); assert_grad(dl, rl, "c4 d_leaves")
    for b in (0, 59, 177):                          # and row by row: no control point hides behind the norm of the others
        assert_grad(dl[b], rl[b], f"c4 d_leaves row {b}"); assert_grad(dj[b], rj[b], f"c4 d_jaws row {b}")


def test_wide_single_pass_variants(torch, monkeypatch):
    """The widest compiled variants (more than 48 KB of shared memory per warp) as ONE pass, including 63, which the default
    splits into 3 x 3 sub-kernels; and the split forced on small kernels."""
    monkeypatch.setenv("PDRT_CONV_SINGLE_MAX", "63")
    wl = W.tiny(seed=13, n_cp=2, kernel_size=5, nx=80, ny=44, nz=76, spacing=3.0, flu=(30, 30))
    eng, orc = pair(wl)
    for k in (47, 55, 63):
        eng.set_kernel_size(k)
        orc.set_kernel_size(k)
        assert eng.info.kernel_passes == 1 and eng.info.kernel_size_compiled >= k
        assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), f"single pass k={k}")
        g = W.seeded_dose_gradient(wl, seed=k)
        dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        assert_grad(dm, rm, f"single pass k={k} d_mu"); assert_grad(dl, rl, f"single pass k={k} d_leaves")
    monkeypatch.setenv("PDRT_CONV_SINGLE_MAX", "5")
    for k in (7, 13, 33):                           # 3 x 3 passes of 5 / 5 / 11 taps
        eng.set_kernel_size(k)
        orc.set_kernel_size(k)
        assert eng.info.kernel_passes == 9
        assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), f"split k={k}")
        g = W.seeded_dose_gradient(wl, seed=k)
        dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        assert_grad(dm, rm, f"split k={k} d_mu"); assert_grad(dl, rl, f"split k={k} d_leaves")


@pytest.mark.parametrize("mode", ["default", "row_symmetric", "output_stationary"])
def test_convolution_kernel_families_on_a_field_wider_than_one_work_item(torch, monkeypatch, mode):
    """The three convolution kernels (k_conv_fold: row + column symmetry, 15..25 taps; k_conv_sym: row symmetry; k_conv:
    output-stationary) on a field so long in v that a slice is split into two work items (chunks along v), forward and adjoint,
    and pdrt_work.conv_symmetric."""
    if mode == "row_symmetric":
        monkeypatch.setenv("PDRT_CONV_FOLD_MAX", "0")
    elif mode == "output_stationary":
        monkeypatch.setenv("PDRT_CONV_LEGACY", "1")
    wl = W.tiny(seed=21, nx=44, ny=40, nz=110, spacing=2.5, n_cp=2, n_pairs=20, kernel_size=21, flu=(24, 110), flu_d=2.5, head_scatter=False)
    eng, orc = pair(wl)
    for k in (21, 11):
        eng.set_kernel_size(k)
        orc.set_kernel_size(k)
        assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), f"{mode} k={k}")
        wf = eng.get_work()
        assert wf.conv_items > 2 * wl.n_cp * eng.info.beam_nw * 0.5 and wf.conv_symmetric == (0 if mode == "output_stationary" else 2 if mode == "default" and k >= 15 else 1)
        g = W.seeded_dose_gradient(wl, seed=k)
        dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        assert_grad(dm, rm, f"{mode} k={k} d_mu"); assert_grad(dl, rl, f"{mode} k={k} d_leaves"); assert_grad(dj, rj, f"{mode} k={k} d_jaws")


@pytest.mark.parametrize("k", [11, 31, 41, 55])
def test_config4_kernel_size_sweep_sampled(torch, k):
    """The other kernel sizes of the c4 sweep at full size, and the paper's operating point k = 55: sampled
    voxels and sampled control points."""
    wl = W.config4(k)
    eng, orc = pair(wl)
    check_sampled_dose(eng, orc, wl, 90, 40 + k, f"c4 k={k}")
    g = W.seeded_dose_gradient(wl, seed=4)
    check_sampled_gradients(eng, orc, wl, g, [5, 120], f"c4 k={k}")


def test_config2_with_head_scatter(torch):
    """Head scatter (two Gaussians) at c2 size: wide blurs over a 110 x 250 mm field, forward and backward."""
    wl = W.config2()
    wl.model.update(n_hs=2, hs_amp=np.asarray([0.04, 0.015], np.float32), hs_sigma_mm=np.asarray([6.0, 14.0], np.float32))
    eng, orc = pair(wl)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "c2+hs dose")
    g = W.seeded_dose_gradient(wl, seed=22)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dm, rm, "c2+hs d_mu"); assert_grad(dj, rj, "c2+hs d_jaws"); assert_grad(dl, rl, "c2+hs d_leaves")


def test_config5_double_arc_sampled(torch):
    """c5: 256x256x160 @ 2 mm, two arcs (356 control points), 80 leaf pairs misaligned with the 2 mm map rows,
    tracking jaws, k = 31: first iteration of the planning loop."""
    wl = W.config5()
    eng, orc = pair(wl)
    check_sampled_dose(eng, orc, wl, 120, 6, "c5")
    g = W.seeded_dose_gradient(wl, seed=6)
    check_sampled_gradients(eng, orc, wl, g, [0, 200, 355], "c5")


# ---------------------------------------------------------------------------------------------------------------
# Code paths the standard cases do not reach
@pytest.mark.parametrize("beam", [
    dict(beam_nu=52, beam_nw=70, beam_du=2.1, beam_dw=1.6, beam_wmin=-55.0),     # finer than the patient grid: > 3 x 3 candidates in S7
    dict(beam_nu=24, beam_nw=20, beam_du=5.5, beam_dw=6.0, beam_wmin=-58.0),     # coarser than the patient grid
], ids=["fine_beam_grid", "coarse_beam_grid"])
def test_beam_grid_that_differs_from_the_patient_grid(torch, beam):
    """Explicit beam grids with du, dw != sx: the general candidate loop of k_resample_adjoint, bilinear stencils that skip
    or repeat beam voxels in k_gather_dose, and map pixels much coarser / finer than beam voxels in S3 / S9."""
    wl = W.tiny(seed=31, nx=30, ny=26, nz=14, spacing=4.0, n_cp=3, kernel_size=7, flu=(22, 18), explicit_beam=beam)
    eng, orc = pair(wl)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "dose")
    g = W.seeded_dose_gradient(wl, seed=31)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dm, rm, "d_mu"); assert_grad(dj, rj, "d_jaws"); assert_grad(dl, rl, "d_leaves")


def test_control_points_in_several_batches(torch, monkeypatch):
    """A scratch cap smaller than the arc (PDRT_SCRATCH_GB) makes the engine run the control points in batches: the
    resampler accumulates into the dose grid across launches and the gradients of later batches use their own blocks."""
    wl = W.tiny(seed=32, n_cp=7, nx=36, ny=30, nz=16, kernel_size=5, flu=(24, 20))
    monkeypatch.setenv("PDRT_SCRATCH_GB", "0.0005")          # room for two or three control points per batch
    eng, orc = pair(wl)
    assert_dose(eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "batched dose")
    g = W.seeded_dose_gradient(wl, seed=32)
    dl, dj, dm = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    assert_grad(dm, rm, "batched d_mu"); assert_grad(dj, rj, "batched d_jaws"); assert_grad(dl, rl, "batched d_leaves")
    n_batches = eng.get_stage_ms()[1]["conv_adj"]
    assert n_batches >= 2, f"expected several batches, got {n_batches} conv launches"


def test_results_are_bit_reproducible(torch):
    """No atomics on the data path and fixed summation orders: two runs give identical bits."""
    wl = W.tiny(seed=33, n_cp=6, nx=40, ny=36, nz=20, kernel_size=9, flu=(28, 24))
    eng, _ = pair(wl)
    g = W.seeded_dose_gradient(wl, seed=33)
    for k in (9, 21, 5):            # row-symmetric, folded (shared-memory ring of output rows) and output-stationary convolution
        eng.set_kernel_size(k)
        d1 = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu).clone()
        b1 = [t.clone() for t in eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)]
        for _ in range(3):
            d2 = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
            b2 = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
            assert torch.equal(d1, d2), f"k={k}"
            assert all(torch.equal(a, b) for a, b in zip(b1, b2)), f"k={k}"


def test_config2_is_bit_reproducible(torch):
    """The same on c2 (k = 21: k_conv_fold, many work items in flight on every SM)."""
    wl = W.config2()
    eng, _ = pair(wl)
    g = W.seeded_dose_gradient(wl, seed=2)
    d1 = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu).clone()
    b1 = [t.clone() for t in eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)]
    for _ in range(3):
        d2 = eng.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
        b2 = eng.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        assert torch.equal(d1, d2)
        assert all(torch.equal(a, b) for a, b in zip(b1, b2))


def test_sharded_driver_around_the_cuda_engine_world_size_1(torch):
    """The per-rank driver of bench.py --gpus N (ShardedDose: Engine + reduce_dose + gather_rows) with a one-rank gloo
    process group on the CUDA engine: the collectives run (trivially) and the results equal the plain calls."""
    import socket
    import torch.distributed as dist
    from paper_2512_18863_b200.shard import ShardedDose
    wl = W.tiny(seed=34, n_cp=5, nx=36, ny=32, nz=16, kernel_size=7, flu=(24, 20))
    eng, orc = pair(wl)
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1)
    try:
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        sh = ShardedDose(eng, t(wl.leaves), t(wl.jaws), t(wl.gantry_deg), t(wl.mu), eng.dose_shape, 0, 1)
        assert (sh.lo, sh.hi) == (0, wl.n_cp)
        assert_dose(sh.forward(), orc.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu), "sharded dose")
        g = W.seeded_dose_gradient(wl, seed=34)
        sh.backward(t(g))
        dl, dj, dm = sh.gather()
        rl, rj, rm = orc.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
        assert_grad(dm, rm, "sharded d_mu"); assert_grad(dj, rj, "sharded d_jaws"); assert_grad(dl, rl, "sharded d_leaves")
    finally:
        dist.destroy_process_group()
