"""Pins of the float64 oracle against what the paper and the mathematics fix.

None of these retypes an oracle formula: they use closed forms, exact invariants, library routines
(scipy.signal, scipy.integrate), brute force and finite differences, chosen so that a dropped term,
a wrong sign or index, or a transposed operand in oracle/pdrt_oracle.c fails at least one of them.
"""
import numpy as np
import pytest
import scipy.integrate
import scipy.signal

from oracle.oracle import Oracle
from paper_2512_18863_b200 import workloads as W


def make(wl):
    return Oracle(wl.grid, wl.model, wl.density)


def water_cube(n=24, s=4.0, k=5, **model_kw):
    """Homogeneous water cube, isocentre at the centre, default beam grid, symmetric leaf bank."""
    grid = W.centred_grid(n, n, n, s)
    model = W.common_model(8, 40.0, 24, 24, s, k)
    model.update(model_kw)
    return grid, model, np.ones((n, n, n), np.float32)


# ----------------------------------------------------------------------------- Eq. 4
def test_eq4_overlap_is_the_pixel_integral_of_the_opening():
    """PAPER.md:105-107 Eq. 4: f = (1/D) * length(pixel ∩ [l,r]); brute-force indicator integral."""
    wl = W.tiny()
    o = make(wl)
    rng = np.random.default_rng(0)
    for _ in range(200):
        c, D = rng.uniform(-20, 20), rng.uniform(0.5, 5)
        lo, hi = np.sort(rng.uniform(c - 2 * D, c + 2 * D, 2))
        x = c - D / 2 + (np.arange(20000) + 0.5) * D / 20000
        brute = np.mean((x > lo) & (x < hi))
        assert abs(o.ov(c, D, lo, hi) - brute) < 1e-4
    assert o.ov(0.0, 2.0, 3.0, -3.0) == 0.0            # l > r: closed
    assert o.ov(0.0, 2.0, -9.0, 9.0) == 1.0            # fully open pixel


def test_eq4_area_conservation_P4():
    """P4: sum_a ov * D = r - l clipped to the map  =>  sum Phi0 * Du * Dv = area(aperture ∩ jaws), tau = 0."""
    wl = W.tiny(seed=11, head_scatter=False)
    wl.model.update(tau=0.0, fwhm_mlc_mm=0.0, fwhm_jaw_mm=0.0, n_oar=0)
    o = make(wl)
    m = wl.model
    for b in range(wl.n_cp):
        _, A, J, P0 = o.fluence(wl.leaves[b], wl.jaws[b], parts=True)
        x1, x2, y1, y2 = [float(v) for v in wl.jaws[b]]
        ulo, uhi = -0.5 * m["flu_nu"] * m["flu_du"], 0.5 * m["flu_nu"] * m["flu_du"]
        vlo, vhi = -0.5 * m["flu_nv"] * m["flu_dv"], 0.5 * m["flu_nv"] * m["flu_dv"]
        area = 0.0
        bounds = np.asarray(m["leaf_bounds_mm"], np.float64)
        for i in range(m["n_pairs"]):
            lu = max(0.0, min(float(wl.leaves[b, 1, i]), x2, uhi) - max(float(wl.leaves[b, 0, i]), x1, ulo))
            lv = max(0.0, min(bounds[i + 1], y2, vhi) - max(bounds[i], y1, vlo))
            area += lu * lv
        # J*A is an area product only where pixels are not cut by both a jaw and a leaf edge; compare the
        # separable parts exactly instead, and the total within one pixel ring.
        assert np.isclose(A.sum() * m["flu_du"] * m["flu_dv"],
                          sum(max(0.0, min(float(wl.leaves[b, 1, i]), uhi) - max(float(wl.leaves[b, 0, i]), ulo)) *
                              max(0.0, min(bounds[i + 1], vhi) - max(bounds[i], vlo)) for i in range(m["n_pairs"])),
                          rtol=1e-12)
        assert np.isclose(J.sum() * m["flu_du"] * m["flu_dv"], (min(x2, uhi) - max(x1, ulo)) * (min(y2, vhi) - max(y1, vlo)), rtol=1e-12)
        ring = 2 * ((x2 - x1) + (y2 - y1)) * max(m["flu_du"], m["flu_dv"])
        assert abs(P0.sum() * m["flu_du"] * m["flu_dv"] - area) <= ring


def test_eq4_subgradients_G9():
    """Away from kinks d ov is the finite difference; at the kinks the half-open convention of G9 holds."""
    o = make(W.tiny())
    rng = np.random.default_rng(1)
    h = 1e-6
    for _ in range(300):
        c, D = rng.uniform(-5, 5), 2.5
        lo, hi = np.sort(rng.uniform(c - 2 * D, c + 2 * D, 2))
        if min(abs(lo - (c - D / 2)), abs(lo - (c + D / 2)), abs(hi - (c - D / 2)), abs(hi - (c + D / 2)), hi - lo) < 1e-3:
            continue
        fd_hi = (o.ov(c, D, lo, hi + h) - o.ov(c, D, lo, hi - h)) / (2 * h)
        fd_lo = (o.ov(c, D, lo + h, hi) - o.ov(c, D, lo - h, hi)) / (2 * h)
        assert abs(o.dov_dhi(c, D, lo, hi) - fd_hi) < 1e-6
        assert abs(o.dov_dlo(c, D, lo, hi) - fd_lo) < 1e-6
    # a closed pair inside a pixel can open: right leaf pulls with +1/D, left leaf with -1/D
    assert o.dov_dhi(0.0, 2.0, 0.3, 0.3) == pytest.approx(0.5)
    assert o.dov_dlo(0.0, 2.0, 0.3, 0.3) == pytest.approx(-0.5)
    # an edge exactly on a pixel boundary belongs to the pixel on its right (hi) / left (lo)
    assert o.dov_dhi(0.0, 2.0, -5.0, -1.0) == pytest.approx(0.5) and o.dov_dhi(0.0, 2.0, -5.0, 1.0) == 0.0
    assert o.dov_dlo(0.0, 2.0, 1.0, 5.0) == pytest.approx(-0.5) and o.dov_dlo(0.0, 2.0, -1.0, 5.0) == 0.0


# ----------------------------------------------------------------------------- Gaussians, off-axis, transmission
def test_gaussian_taps_and_blur_against_scipy():
    """G13: normalised taps out to ceil(3 sigma / D); the blur is scipy's zero-padded 'same' convolution."""
    o = make(W.tiny())
    T, g = o.gauss_taps(1.7, 2.5)
    assert T == 3 and len(g) == 7 and np.isclose(g.sum(), 1.0) and np.allclose(g, g[::-1])
    assert np.isclose(g[T + 1] / g[T], np.exp(-2.5 ** 2 / (2 * 1.7 ** 2)))
    assert o.gauss_taps(0.0, 2.5)[0] == 0
    # FWHM: the continuous Gaussian falls to one half at FWHM/2
    fwhm = 4.0
    sigma = fwhm / 2.354820045
    assert np.isclose(np.exp(-(fwhm / 2) ** 2 / (2 * sigma ** 2)), 0.5, atol=1e-9)
    a = np.random.default_rng(2).standard_normal((9, 13))
    assert np.allclose(o.blur_axis(a, 0, T, g), scipy.signal.convolve2d(a, g[None, :], mode="same"))
    assert np.allclose(o.blur_axis(a, 1, T, g), scipy.signal.convolve2d(a, g[:, None], mode="same"))


def test_fluence_corrections_compose_as_stated():
    """O2-O5 special cases: open field => J; closed leaves => tau*J; OAR multiplies; head scatter adds
    amp * (blurred Phi0); blur of a wide-open field leaves the interior untouched."""
    wl = W.tiny(seed=3, head_scatter=False)
    m = wl.model
    m.update(fwhm_mlc_mm=0.0, fwhm_jaw_mm=0.0, n_oar=0, tau=0.01)
    np_ = m["n_pairs"]
    jaws = np.array([-12.0, 15.0, -10.0, 9.0])
    open_leaves = np.stack([np.full(np_, -500.0), np.full(np_, 500.0)])
    closed = np.zeros((2, np_))
    o = make(wl)
    P_open, A, J, _ = o.fluence(open_leaves, jaws, parts=True)
    rows_in_bank = A.max(axis=1) > 0
    assert np.allclose(P_open[rows_in_bank], J[rows_in_bank] * (0.01 + 0.99 * A[rows_in_bank]))
    assert np.allclose(o.fluence(closed, jaws), 0.01 * J)
    # off-axis: radial table, linear interpolation, clamped
    m2 = dict(m, n_oar=3, oar_dr_mm=10.0, oar=np.array([1.0, 2.0, 4.0], np.float32))
    P_oar = Oracle(wl.grid, m2, wl.density).fluence(open_leaves, jaws)
    uf = (np.arange(m["flu_nu"]) - 0.5 * (m["flu_nu"] - 1)) * m["flu_du"]
    vf = (np.arange(m["flu_nv"]) - 0.5 * (m["flu_nv"] - 1)) * m["flu_dv"]
    r = np.hypot(uf[None, :], vf[:, None])
    assert np.allclose(P_oar, P_open * np.interp(r, [0.0, 10.0, 20.0], [1.0, 2.0, 4.0]))
    # head scatter: a single Gaussian of amplitude 0.1 adds 0.1 * (2-D Gaussian blur of Phi0)
    m3 = dict(m, n_hs=1, hs_amp=np.array([0.1], np.float32), hs_sigma_mm=np.array([5.0], np.float32))
    o3 = Oracle(wl.grid, m3, wl.density)
    Tu, gu = o3.gauss_taps(5.0, m["flu_du"])
    Tv, gv = o3.gauss_taps(5.0, m["flu_dv"])
    blurred = scipy.signal.convolve2d(P_open, np.outer(gv, gu), mode="same")
    assert np.allclose(o3.fluence(open_leaves, jaws), P_open + 0.1 * blurred)
    # penumbra: u-blur uses the MLC FWHM, v-blur the jaw FWHM (distinguishable by their widths)
    m4 = dict(m, fwhm_mlc_mm=3.0, fwhm_jaw_mm=7.0)
    o4 = Oracle(wl.grid, m4, wl.density)
    _, gu = o4.gauss_taps(3.0 / 2.354820045, m["flu_du"])
    _, gv = o4.gauss_taps(7.0 / 2.354820045, m["flu_dv"])
    assert np.allclose(o4.fluence(open_leaves, jaws), scipy.signal.convolve2d(P_open, np.outer(gv, gu), mode="same"))


# ----------------------------------------------------------------------------- P5 radiological depth
def test_radiological_depth_water_and_slabs_P5():
    """Eq. 7 closed forms: water box => geometric depth below the surface; y-normal slabs at gantry 0 =>
    sum rho_i t_i (exact one voxel away from a slab face, within 0.3125*|d rho| mm next to it: the trilinear
    ramp between two voxel centres integrates to the sharp-face value only once fully traversed)."""
    wl = W.config2()
    o = make(wl)
    ny, s = wl.grid["ny"], wl.grid["sy"]
    depth = (np.arange(ny) + 0.5) * s                      # slice k sits at voxel-centre depth (default beam grid)
    sharp = np.zeros(ny)
    for k, d in enumerate(depth):
        t = np.linspace(0, d, 200001)
        rho = np.where((t >= 40) & (t < 70), 0.25, np.where((t >= 100) & (t < 120), 1.8, 1.0))
        sharp[k] = np.trapezoid(rho, t)
    z = o.radiological_depth(0.0)
    near = np.zeros(ny, bool)
    for face in (40, 70, 100, 120):
        near |= np.abs(depth - face) < s
    assert np.allclose(z[~near], sharp[~near], atol=2e-3)
    assert np.all(np.abs(z[near] - sharp[near]) <= 0.3125 * 1.55 + 2e-3)
    # gantry 180: the same slabs are traversed from the posterior side
    z180 = o.radiological_depth(180.0)
    total = sharp[-1] + 1.0 * 0.5 * s                      # full traversal = 128 voxels
    assert np.isclose(z180[-1], total - (sharp[0] - 0.0) + 0.0, atol=0.5)
    # water: radiological depth == geometric depth, at any angle while the ray is inside the box
    ow = Oracle(wl.grid, wl.model, np.ones_like(wl.density))
    assert np.allclose(ow.radiological_depth(0.0), depth, atol=1e-9)
    for phi in (30.0, 72.0, 200.0):
        c, sn = np.cos(np.radians(phi)), np.sin(np.radians(phi))
        half = 0.5 * ny * s
        entry = min(half / abs(c) if abs(c) > 1e-12 else np.inf, half / abs(sn) if abs(sn) > 1e-12 else np.inf)
        w = (np.arange(ny) - 0.5 * (ny - 1)) * s
        expect = np.clip(w + entry, 0.0, 2 * entry)
        zphi = ow.radiological_depth(phi)
        # the entry point falls inside a sampling interval: the midpoint rule is off by at most ds/2 there,
        # and exact (slope 1 in water) from then on
        assert np.all(np.abs(zphi - expect) <= 0.5 * 1.25 + 1e-9)
        inside = (expect > 2.5) & (expect < 2 * entry - 2.5)
        assert np.allclose(np.diff(zphi[inside]), s, atol=1e-9)


def test_radiological_depth_oblique_slabs_and_rotation_sense():
    """Oblique ray through y-normal slabs: thicknesses scale with 1/|cos phi|; and the rotation sense of
    reading G1: at gantry 90 the source sits on the +x side."""
    wl = W.config2()
    o = make(wl)
    phi = 25.0
    c = np.cos(np.radians(phi))
    z = o.radiological_depth(phi)
    half = 0.5 * wl.grid["ny"] * wl.grid["sy"]
    w = (np.arange(wl.grid["ny"]) - 0.5 * (wl.grid["ny"] - 1)) * wl.grid["sy"]
    path = w + half / c                                    # path length inside the box (enters through the -y face)
    ydepth = path * c
    expect = np.array([np.trapezoid(np.where((t >= 40) & (t < 70), 0.25, np.where((t >= 100) & (t < 120), 1.8, 1.0)), t) / c
                       for t in (np.linspace(0, d, 100001) for d in ydepth)])
    assert np.allclose(z, expect, atol=0.3125 * 1.55 / c + 0.5 * 1.25 * 1.8 + 0.05)
    # rotation sense: dense half-space x > 0
    grid = W.centred_grid(32, 32, 8, 2.5)
    Z, Y, X = W.voxel_coords(grid)
    rho = np.where(X > 0, 2.0, 0.5).astype(np.float32)
    m = W.common_model(8, 20.0, 16, 16, 2.5, 3)
    oh = Oracle(grid, m, rho)
    z90, z270 = oh.radiological_depth(90.0), oh.radiological_depth(270.0)
    k_iso = 15                                            # w = -1.25 mm: just before the isocentre plane
    assert np.isclose(z90[k_iso], 2.0 * (40.0 - 1.25), atol=1.0)      # came through the dense side
    assert np.isclose(z270[k_iso], 0.5 * (40.0 - 1.25), atol=1.0)


# ----------------------------------------------------------------------------- P7 kernel table
def test_kernel_table_against_polar_quadrature_P7():
    """sum W_tab over the k x k window vs the integral of K over the same square, done in polar coordinates
    (the 1/r cancels against the Jacobian):  ∫_0^2π F(R(θ)) dθ, F(R) = A(1-e^{-aR})/a + B(1-e^{-bR})/b."""
    grid, model, rho = water_cube(n=12, s=2.5, k=9)
    sums = []
    for k in (5, 9, 15):
        model["kernel_size"] = k
        o = Oracle(grid, model, rho)
        Wt = o.kernel_table()
        assert Wt.shape == (model["n_z"], k, k)
        assert np.allclose(Wt, Wt[:, ::-1, :]) and np.allclose(Wt, Wt[:, :, ::-1]) and np.allclose(Wt, Wt.transpose(0, 2, 1))
        half = 0.5 * k * 2.5
        for n in (1, 20, 100):
            A, a, B, b = (float(model[key][n]) for key in ("kA", "ka", "kB", "kb"))
            F = lambda R: A * (1 - np.exp(-a * R)) / a + B * (1 - np.exp(-b * R)) / b
            square = lambda hh: 8 * scipy.integrate.quad(lambda th: F(hh / np.cos(th)), 0, np.pi / 4, epsabs=1e-13)[0]
            exact, centre = square(half), square(0.5 * 2.5)
            assert abs(Wt[n].sum() - exact) / exact < 0.04       # 8x8 midpoint rule on the 1/r singularity
            c = (k - 1) // 2                                     # away from the singular pixel the rule is tight
            assert abs((Wt[n].sum() - Wt[n, c, c]) - (exact - centre)) / (exact - centre) < 5e-3
        sums.append(Wt[50].sum())
    assert sums[0] < sums[1] < sums[2]
    # linear interpolation between nodes (G5), clamped at both ends
    assert np.allclose(o.slice_kernel(Wt, 3.0), 0.5 * (Wt[1] + Wt[2]))
    assert np.allclose(o.slice_kernel(Wt, -4.0), Wt[0]) and np.allclose(o.slice_kernel(Wt, 1e6), Wt[-1])


# ----------------------------------------------------------------------------- P6 convolution
def test_convolution_against_scipy_and_delta_P6():
    """Eq. 8 per slice vs scipy.signal.correlate2d (zero-padded 'same'); a delta returns the kernel itself;
    a uniform field wider than the kernel returns Phi * sum W at the centre."""
    wl = W.tiny(seed=5, nx=14, ny=6, nz=11, kernel_size=7, n_cp=1)
    o = make(wl)
    Wt = o.kernel_table()
    rng = np.random.default_rng(5)
    Nw, Nv, Nu = o.beam_shape
    P = rng.standard_normal(o.beam_shape)
    z = rng.uniform(0, 300, Nw)
    D = o.convolve(Wt, z, P)
    for k in range(Nw):
        Wk = o.slice_kernel(Wt, z[k])
        assert np.allclose(D[k], scipy.signal.correlate2d(P[k], Wk, mode="same"), atol=1e-12)
    delta = np.zeros(o.beam_shape)
    delta[:, 5, 7] = 1.0
    Dd = o.convolve(Wt, z, delta)
    Wk = o.slice_kernel(Wt, z[2])
    assert np.allclose(Dd[2, 2:9, 4:11], Wk[::-1, ::-1]) and np.allclose(Wk, Wk[::-1, ::-1])
    ones = np.ones(o.beam_shape)
    assert np.isclose(o.convolve(Wt, z, ones)[3, 5, 7], o.slice_kernel(Wt, z[3]).sum())


# ----------------------------------------------------------------------------- P9 projection
def test_projection_magnification_and_inverse_square_P9():
    """Eq. 5-6: at the isocentre plane (d = SID) the fluence map is reproduced sample for sample; off it the
    pattern is magnified by d/SID and scaled by (SID/d)^2 so that fluence x area is conserved."""
    grid = W.centred_grid(40, 41, 16, 2.5)                # odd Nw: slice 20 sits exactly at w = 0
    model = W.common_model(8, 20.0, 40, 16, 2.5, 3)
    o = Oracle(grid, model, np.ones((16, 41, 40), np.float32))
    Phimap = np.random.default_rng(6).uniform(0.5, 1.5, (16, 40))
    Phimap[:, :8] = Phimap[:, -8:] = 0.0
    Phimap[:3] = Phimap[-3:] = 0.0
    V = o.project(Phimap)
    assert np.allclose(V[20], Phimap)                     # w = 0, mag = 1, same grids
    for k in (0, 40):
        d = 1000.0 + (k - 20) * 2.5
        assert np.isclose(V[k].sum() * 2.5 * 2.5, Phimap.sum() * 2.5 * 2.5, rtol=2e-2)
    # a single bright pixel at u = +21.25 mm lands at u * d/SID, with weight (SID/d)^2
    spot = np.zeros((16, 40))
    spot[8, 28] = 1.0                                     # uf = (28 - 19.5)*2.5 = 21.25, vf = +1.25
    Vs = o.project(spot)
    u = (np.arange(40) - 19.5) * 2.5
    for k in (4, 36):
        d = 1000.0 + (k - 20) * 2.5
        centroid = (Vs[k].sum(axis=0) * u).sum() / Vs[k].sum()
        assert np.isclose(centroid, 21.25 * d / 1000.0, atol=0.05)
        assert np.isclose(Vs[k].sum(), (1000.0 / d) ** 2 * (d / 1000.0) ** 2, rtol=0.02)   # mag^2 x (footprint / mag^2)


# ----------------------------------------------------------------------------- P8 resampling
def test_resample_identity_and_quarter_turns_P8():
    """Gantry 0 with beam grid == patient grid: the resampler is the identity (config 1 geometry).  Gantry
    90/180/270 on a cubic isotropic water grid centred on the isocentre: exact axis permutations/flips."""
    wl = W.config1()
    wl.grid.update(nx=20, ny=20, nz=20, ox=-23.75, oy=1.25, oz=-23.75)
    wl.model.update(beam_nu=20, beam_nw=20, flu_nu=20, flu_nv=20, n_pairs=8,
                    leaf_bounds_mm=np.linspace(-20, 20, 9).astype(np.float32), kernel_size=5)
    o = Oracle(wl.grid, wl.model, np.ones((20, 20, 20), np.float32))
    Db = np.random.default_rng(8).standard_normal(o.beam_shape)
    dose = o.resample_add(0.0, 2.0, Db)
    assert np.array_equal(dose, 2.0 * Db.transpose(1, 0, 2))       # [w][v][u] -> [z][y][x]
    grid, model, rho = water_cube()
    oc = Oracle(grid, model, rho)
    leaves = np.stack([np.linspace(-30, -6, 8), np.linspace(4, 28, 8)])     # asymmetric on purpose
    jaws = np.array([-25.0, 20.0, -18.0, 22.0])
    d0 = oc.dose(leaves[None], jaws[None], [0.0], [1.0])
    d90 = oc.dose(leaves[None], jaws[None], [90.0], [1.0])
    d180 = oc.dose(leaves[None], jaws[None], [180.0], [1.0])
    d270 = oc.dose(leaves[None], jaws[None], [270.0], [1.0])
    assert d0.max() > 0
    tol = 1e-9 * d0.max()
    assert np.allclose(d90, d0.transpose(0, 2, 1)[:, :, ::-1], atol=tol)       # (x,y) <- (u=y, w=-x)
    assert np.allclose(d180, d0[:, ::-1, ::-1], atol=tol)
    assert np.allclose(d270, d0.transpose(0, 2, 1)[:, ::-1, :], atol=tol)
    # source side (G1): at gantry 0 the beam travels +y, so dose builds up from the -y face
    prof = d0[12, :, 12]
    assert prof[1] > prof[0] and prof[-1] < prof.max()


# ----------------------------------------------------------------------------- P1, P2, P3 whole path
def test_mu_linearity_and_arc_additivity_P1():
    wl = W.tiny(seed=21)
    o = make(wl)
    d = o.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    assert np.allclose(o.dose(wl.leaves, wl.jaws, wl.gantry_deg, 2.5 * wl.mu.astype(np.float64)), 2.5 * d, rtol=1e-13)
    parts = sum(o.dose(wl.leaves[b:b + 1], wl.jaws[b:b + 1], wl.gantry_deg[b:b + 1], wl.mu[b:b + 1]) for b in range(wl.n_cp))
    assert np.allclose(parts, d, rtol=1e-12, atol=1e-15)
    Db = o.beam_dose(wl.leaves[0], wl.jaws[0], wl.gantry_deg[0])
    single = o.resample_add(wl.gantry_deg[0], wl.model["cal"] * float(wl.mu[0]), Db)
    assert np.allclose(single, o.dose(wl.leaves[:1], wl.jaws[:1], wl.gantry_deg[:1], wl.mu[:1]), rtol=1e-13)


def test_closed_aperture_gives_zero_dose_P2():
    wl = W.tiny(seed=22)
    o = make(wl)
    jaws = wl.jaws.copy()
    jaws[:, 1] = jaws[:, 0]
    assert np.all(o.dose(wl.leaves, jaws, wl.gantry_deg, wl.mu) == 0.0)
    wl.model["tau"] = 0.0
    o0 = make(wl)
    closed = np.zeros_like(wl.leaves)
    assert np.all(o0.dose(closed, wl.jaws, wl.gantry_deg, wl.mu) == 0.0)
    assert o.dose(closed, wl.jaws, wl.gantry_deg, wl.mu).max() > 0.0      # transmission leaks with tau > 0


def test_mirror_symmetry_in_water_P3():
    grid, model, rho = water_cube()
    o = Oracle(grid, model, rho)
    right = np.array([5.0, 11.0, 17.0, 23.0, 23.0, 17.0, 11.0, 5.0])       # symmetric in i
    leaves = np.stack([-right, right])
    jaws = np.array([-26.0, 26.0, -30.0, 30.0])
    d = o.dose(leaves[None], jaws[None], [0.0], [3.0])
    assert d.max() > 0
    assert np.allclose(d, d[:, :, ::-1], rtol=1e-10, atol=1e-14 * d.max())      # u -> -u
    assert np.allclose(d, d[::-1, :, :], rtol=1e-10, atol=1e-14 * d.max())      # v -> -v


def test_calibration_identity_P12():
    """scale so a reference MU gives 1 Gy at 10x10 cm, 10 cm depth, SSD 90 cm in water."""
    s = 5.0
    grid = dict(nx=40, ny=40, nz=40, sx=s, sy=s, sz=s, ox=-97.5, oy=-97.5, oz=-97.5, iso=(0.0, 0.0, 0.0))
    model = W.common_model(40, 100.0, 40, 40, s, 9)        # iso 100 mm below the -y face: SSD = 900 mm
    o = Oracle(grid, model, np.ones((40, 40, 40), np.float32))
    leaves = np.stack([np.full(40, -100.0), np.full(40, 100.0)])[None]
    jaws = np.array([[-50.0, 50.0, -50.0, 50.0]])
    ref = [19, 19, 19]                                     # nearest voxel to the isocentre
    d_ref = o.dose_at(leaves, jaws, [0.0], [100.0], [ref])[0]
    model2 = dict(model, cal=model["cal"] / d_ref)
    o2 = Oracle(grid, model2, np.ones((40, 40, 40), np.float32))
    assert np.isclose(o2.dose(leaves, jaws, [0.0], [100.0])[19, 19, 19], 1.0, rtol=1e-12)


def test_dose_at_matches_full_dose():
    wl = W.tiny(seed=23)
    o = make(wl)
    d = o.dose(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu)
    rng = np.random.default_rng(23)
    ijk = np.stack([rng.integers(0, wl.grid["nx"], 40), rng.integers(0, wl.grid["ny"], 40), rng.integers(0, wl.grid["nz"], 40)], axis=1)
    got = o.dose_at(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, ijk)
    assert np.allclose(got, d[ijk[:, 2], ijk[:, 1], ijk[:, 0]], rtol=1e-11, atol=1e-16)


# ----------------------------------------------------------------------------- P10, P11 adjoint
def test_adjoint_identities_P10():
    """<A x, y> = <x, A^T y> to rounding for every linear stage."""
    wl = W.tiny(seed=31)
    o = make(wl)
    rng = np.random.default_rng(31)
    Wt = o.kernel_table()
    z = o.radiological_depth(wl.gantry_deg[0])
    x = rng.standard_normal(o.flu_shape)
    y = rng.standard_normal(o.beam_shape)
    assert np.isclose((o.project(x) * y).sum(), (x * o.project_adjoint(y)).sum(), rtol=1e-12)
    x = rng.standard_normal(o.beam_shape)
    assert np.isclose((o.convolve(Wt, z, x) * y).sum(), (x * o.convolve(Wt, z, y, transpose=True)).sum(), rtol=1e-12)
    g = rng.standard_normal(o.dose_shape).astype(np.float32)
    for phi in (0.0, 33.0, 90.0, 217.5):
        lhs = (o.resample_add(phi, 1.0, x) * g).sum()
        assert np.isclose(lhs, (x * o.resample_adjoint(phi, g)).sum(), rtol=1e-12)
    T, gt = o.gauss_taps(2.2, 3.0)
    a, b = rng.standard_normal(o.flu_shape), rng.standard_normal(o.flu_shape)
    for axis in (0, 1):
        assert np.isclose((o.blur_axis(a, axis, T, gt) * b).sum(), (a * o.blur_axis(b, axis, T, gt, transpose=True)).sum(), rtol=1e-12)


def _nudge_off_kinks(wl, min_dist=0.05):
    """Move leaf and jaw edges at least min_dist away from every pixel boundary and from each other."""
    m = wl.model
    for arr, D, n in ((wl.leaves, m["flu_du"], m["flu_nu"]), (wl.jaws[:, :2], m["flu_du"], m["flu_nu"]), (wl.jaws[:, 2:], m["flu_dv"], m["flu_nv"])):
        edge0 = -0.5 * n * D
        frac = (arr.astype(np.float64) - edge0) / D
        off = frac - np.round(frac)
        bad = np.abs(off) < min_dist / D
        arr[bad] += np.float32(2 * min_dist)
    return wl


def test_gradients_against_central_differences_P11():
    """dL/d(leaves, jaws, MU) for L = <g, dose> vs central finite differences in float64 (h = 1e-3):
    the dose is piecewise linear in leaves/jaws and linear in MU, so FD is exact to rounding off the kinks."""
    wl = _nudge_off_kinks(W.tiny(seed=41, n_cp=2))
    o = make(wl)
    rng = np.random.default_rng(41)
    g = rng.standard_normal(o.dose_shape).astype(np.float32)
    lv, jw, mu = wl.leaves.astype(np.float64), wl.jaws.astype(np.float64), wl.mu.astype(np.float64)
    dl, dj, dm = o.dose_backward(lv, jw, wl.gantry_deg, mu, g)
    L = lambda l_, j_, m_: float((o.dose(l_, j_, wl.gantry_deg, m_) * g).sum())
    h = 1e-3
    scale = max(np.abs(dl).max(), np.abs(dj).max())
    assert scale > 0
    for b in range(wl.n_cp):
        e = np.zeros_like(mu); e[b] = h
        assert np.isclose(dm[b], (L(lv, jw, mu + e) - L(lv, jw, mu - e)) / (2 * h), rtol=1e-7)
        for q in range(4):
            e = np.zeros_like(jw); e[b, q] = h
            fd = (L(lv, jw + e, mu) - L(lv, jw - e, mu)) / (2 * h)
            assert abs(dj[b, q] - fd) <= 1e-6 * scale, (b, q, dj[b, q], fd)
        for bank in range(2):
            for i in range(wl.model["n_pairs"]):
                e = np.zeros_like(lv); e[b, bank, i] = h
                fd = (L(lv + e, jw, mu) - L(lv - e, jw, mu)) / (2 * h)
                assert abs(dl[b, bank, i] - fd) <= 1e-6 * scale, (b, bank, i, dl[b, bank, i], fd)
    assert np.count_nonzero(dl) > wl.model["n_pairs"]       # the check is not vacuous


def test_mu_gradient_is_the_beam_dose_inner_product():
    """d_mu_b = <g, cal R_b D_b> (closed form from Eq. 9's linearity)."""
    wl = W.tiny(seed=42)
    o = make(wl)
    g = np.random.default_rng(42).standard_normal(o.dose_shape).astype(np.float32)
    _, _, dm = o.dose_backward(wl.leaves, wl.jaws, wl.gantry_deg, wl.mu, g)
    for b in range(wl.n_cp):
        one = o.dose(wl.leaves[b:b + 1], wl.jaws[b:b + 1], wl.gantry_deg[b:b + 1], [1.0])
        assert np.isclose(dm[b], (one * g).sum(), rtol=1e-11)
