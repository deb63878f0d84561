"""Seeded synthetic workloads — inputs only.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic: it only draws seeded random numbers (numpy PCG64), paints phantoms and fills the
plain-dict mirrors of `pdrt_grid` / `pdrt_beam_model` (include/pdrt.h).  The paper's workloads
are clinical prostate VMAT plans on CTs that are not available; these inputs
take their shapes (≈5 M-voxel pelvis grid at 2-2.5 mm, 178 control points per arc, 5 mm leaves,
kernel 11-41 px) and stand in for them.

Every array is float32, C-contiguous.  Layouts: density [nz][ny][nx]; leaves [n_cp][2][Np]
(bank 0 = left, bank 1 = right); jaws [n_cp][4] = x1,x2,y1,y2; gantry_deg [n_cp]; mu [n_cp].
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SID_MM = 1000.0


@dataclass
class Workload:
    name: str
    seed: int
    grid: dict
    model: dict
    density: np.ndarray
    leaves: np.ndarray
    jaws: np.ndarray
    gantry_deg: np.ndarray
    mu: np.ndarray
    backward: bool = False
    kernel_sizes: tuple = ()
    masks: dict = field(default_factory=dict)   # name -> (bool [nz][ny][nx], weight, prescribed dose or None)

    @property
    def n_cp(self) -> int:
        return int(self.gantry_deg.shape[0])


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def common_model(n_pairs: int, leaf_half_extent: float, flu_nu: int, flu_nv: int, flu_d: float,
                 kernel_size: int) -> dict:
    """The common synthetic beam model of SURVEY.md §8(d).  The kernel parameter tables are this
    build's invention (closed forms below), NOT the coefficients of the paper's ref. [17]."""
    z = np.arange(256, dtype=np.float64) * 2.0
    mu_att = 0.004
    P = (1.0 - np.exp(-0.25 * z)) * np.exp(-mu_att * z)
    S = 0.35 * (1.0 - np.exp(-0.01 * z)) * np.exp(-mu_att * z)
    a = 0.30 - 2e-4 * z
    b = 0.030 - 2e-5 * z
    r = np.arange(0.0, 300.0 + 1e-9, 5.0)
    return dict(
        sid_mm=SID_MM, n_pairs=n_pairs,
        leaf_bounds_mm=_f32(np.linspace(-leaf_half_extent, leaf_half_extent, n_pairs + 1)),
        flu_nu=flu_nu, flu_nv=flu_nv, flu_du=flu_d, flu_dv=flu_d,
        tau=0.002, fwhm_mlc_mm=3.0, fwhm_jaw_mm=4.0,
        n_hs=0, hs_amp=_f32([]), hs_sigma_mm=_f32([]),
        n_oar=len(r), oar_dr_mm=5.0, oar=_f32(1.0 + 0.03 * (r / 100.0) ** 2),
        n_z=256, dz_mm=2.0,
        kA=_f32(P * a / (2 * np.pi)), ka=_f32(a), kB=_f32(S * b / (2 * np.pi)), kb=_f32(b),
        kernel_size=kernel_size, cal=0.01,
        beam_nu=0, beam_nw=0, beam_du=0.0, beam_dw=0.0, beam_wmin=0.0,   # 0 => default beam grid
        ray_step_mm=0.0,                                                   # 0 => 0.5 * min spacing
    )


def centred_grid(nx, ny, nz, s) -> dict:
    """Grid with the isocentre (0,0,0) at its geometric centre."""
    return dict(nx=nx, ny=ny, nz=nz, sx=s, sy=s, sz=s,
                ox=-0.5 * (nx - 1) * s, oy=-0.5 * (ny - 1) * s, oz=-0.5 * (nz - 1) * s, iso=(0.0, 0.0, 0.0))


def voxel_coords(grid):
    x = grid["ox"] + np.arange(grid["nx"]) * grid["sx"]
    y = grid["oy"] + np.arange(grid["ny"]) * grid["sy"]
    z = grid["oz"] + np.arange(grid["nz"]) * grid["sz"]
    return np.meshgrid(z, y, x, indexing="ij")   # each [nz][ny][nx]: Z, Y, X


def _ellipsoid(Z, Y, X, centre, semi):
    return ((X - centre[0]) / semi[0]) ** 2 + ((Y - centre[1]) / semi[1]) ** 2 + ((Z - centre[2]) / semi[2]) ** 2 <= 1.0


# ----------------------------------------------------------------------------- c1
def config1() -> Workload:
    """Water phantom 64^3 @ 2.5 mm, one beam at gantry 0, SSD = SID = 100 cm, 10x10 cm jaws,
    40 retracted leaf pairs, MU 100, fluence 64x64, k = 11.  Beam grid == patient grid."""
    s = 2.5
    grid = dict(nx=64, ny=64, nz=64, sx=s, sy=s, sz=s, ox=-78.75, oy=1.25, oz=-78.75, iso=(0.0, 0.0, 0.0))
    model = common_model(40, 100.0, 64, 64, s, 11)
    model.update(beam_nu=64, beam_nw=64, beam_du=s, beam_dw=s, beam_wmin=1.25)
    leaves = np.zeros((1, 2, 40), np.float32)
    leaves[:, 0, :] = -100.0
    leaves[:, 1, :] = 100.0
    return Workload("c1", 1001, grid, model, np.ones((64, 64, 64), np.float32), leaves,
                    _f32([[-50, 50, -50, 50]]), _f32([0.0]), _f32([100.0]), kernel_sizes=(11,))


# ----------------------------------------------------------------------------- c2
def config2() -> Workload:
    """Slab phantom 128x128x96 @ 2.5 mm, 5 static beams, 60 pairs with irregular apertures, k = 21."""
    rng = np.random.Generator(np.random.PCG64(1002))
    grid = centred_grid(128, 128, 96, 2.5)
    Z, Y, X = voxel_coords(grid)
    depth = Y - (grid["oy"] - 0.5 * grid["sy"])          # from the anterior (-y) face
    rho = np.ones_like(depth)
    rho[(depth >= 40) & (depth < 70)] = 0.25             # lung slab, 3 cm
    rho[(depth >= 100) & (depth < 120)] = 1.8            # bone slab, 2 cm
    model = common_model(60, 150.0, 64, 128, 2.5, 21)
    n_cp = 5
    draws = rng.uniform(-50.0, 50.0, size=(n_cp, 2, 60))
    leaves = np.stack([draws.min(axis=1), draws.max(axis=1)], axis=1)
    jaws = np.tile([-55.0, 55.0, -125.0, 125.0], (n_cp, 1))
    mu = rng.uniform(50.0, 150.0, size=n_cp)
    return Workload("c2", 1002, grid, model, _f32(rho), _f32(leaves), _f32(jaws),
                    _f32([0, 72, 144, 216, 288]), _f32(mu), kernel_sizes=(21,))


# ----------------------------------------------------------------------------- c3..c5 phantom
def pelvis_phantom(grid, rng) -> np.ndarray:
    """Synthetic prostate CT: air, body ellipse 36x22 cm, pelvic-bone ellipsoids, rectal air pocket."""
    Z, Y, X = voxel_coords(grid)
    rho = np.full(Z.shape, 0.001)
    body = (X / 180.0) ** 2 + (Y / 110.0) ** 2 <= 1.0
    noise = rng.standard_normal(Z.shape)
    rho[body] = 1.0 + 0.02 * noise[body]
    for centre, semi in (((-90.0, 10.0, 0.0), (30.0, 35.0, 45.0)), ((90.0, 10.0, 0.0), (30.0, 35.0, 45.0)),
                         ((0.0, 70.0, 0.0), (40.0, 20.0, 50.0))):
        rho[_ellipsoid(Z, Y, X, centre, semi)] = rng.uniform(1.6, 1.9)
    rho[_ellipsoid(Z, Y, X, (0.0, 45.0, 0.0), (15.0, 12.0, 30.0))] = 0.001
    return _f32(rho)


def pelvis_masks(grid) -> dict:
    """Target / OAR masks of the quadratic objective: name -> (mask, weight, prescription)."""
    Z, Y, X = voxel_coords(grid)
    return {
        "target": (_ellipsoid(Z, Y, X, (0, 0, 0), (25, 25, 25)), 100.0, 3.0),
        "bladder": (_ellipsoid(Z, Y, X, (0, -45, 0), (30, 25, 30)), 1.0, None),
        "rectum": (_ellipsoid(Z, Y, X, (0, 45, 0), (20, 17, 35)), 10.0, None),
    }


def _target_leaves(rng, n_cp, bounds, closed_gap):
    """Leaf gaps 0-4 cm around the projection of a 5 cm spherical target; other pairs closed."""
    n_pairs = len(bounds) - 1
    centre_v = 0.5 * (bounds[:-1] + bounds[1:])
    open_pair = np.abs(centre_v) < 25.0
    c = rng.normal(0.0, 3.0, size=(n_cp, n_pairs))
    gap = rng.uniform(0.0, 40.0, size=(n_cp, n_pairs))
    left = np.where(open_pair, c - 0.5 * gap, -0.5 * closed_gap)
    right = np.where(open_pair, c + 0.5 * gap, 0.5 * closed_gap)
    return np.stack([left, right], axis=1), open_pair


def config3() -> Workload:
    """Prostate CT 200x200x120 @ 2.5 mm, one 360-degree arc of 178 control points, 60 pairs, k = 21, forward."""
    rng = np.random.Generator(np.random.PCG64(1003))
    grid = centred_grid(200, 200, 120, 2.5)
    rho = pelvis_phantom(grid, rng)
    model = common_model(60, 150.0, 64, 128, 2.5, 21)
    n_cp = 178
    gantry = (181.0 + 2.0 * np.arange(n_cp)) % 360.0
    leaves, _ = _target_leaves(rng, n_cp, np.asarray(model["leaf_bounds_mm"], np.float64), 0.0)
    jaws = np.tile([-35.0, 35.0, -30.0, 30.0], (n_cp, 1))
    mu = rng.uniform(1.0, 4.0, size=n_cp)
    return Workload("c3", 1003, grid, model, rho, _f32(leaves), _f32(jaws), _f32(gantry), _f32(mu), kernel_sizes=(21,))


def config4(kernel_size: int = 21) -> Workload:
    """Same CT and arc, 80 pairs, fluence 64x160, closed pairs keep a 0.5 mm gap; forward + backward;
    kernel-size sweep 11/21/31/41."""
    rng = np.random.Generator(np.random.PCG64(1004))
    grid = centred_grid(200, 200, 120, 2.5)
    rho = pelvis_phantom(grid, rng)
    model = common_model(80, 200.0, 64, 160, 2.5, kernel_size)
    n_cp = 178
    gantry = (181.0 + 2.0 * np.arange(n_cp)) % 360.0
    leaves, _ = _target_leaves(rng, n_cp, np.asarray(model["leaf_bounds_mm"], np.float64), 0.5)
    jaws = np.tile([-35.0, 35.0, -30.0, 30.0], (n_cp, 1))
    mu = rng.uniform(1.0, 4.0, size=n_cp)
    return Workload("c4", 1004, grid, model, rho, _f32(leaves), _f32(jaws), _f32(gantry), _f32(mu),
                    backward=True, kernel_sizes=(11, 21, 31, 41), masks=pelvis_masks(grid))


def track_jaws(leaves, bounds, margin=5.0, min_gap=1e-6):
    """Jaws tracking the aperture: x1 = min l - 5, x2 = max r + 5 over open pairs; y1/y2 = their v-extent."""
    n_cp = leaves.shape[0]
    jaws = np.zeros((n_cp, 4))
    for b in range(n_cp):
        open_pair = (leaves[b, 1] - leaves[b, 0]) > 0.6       # wider than the 0.5 mm parked gap
        if not open_pair.any():
            open_pair[:] = True
        idx = np.nonzero(open_pair)[0]
        jaws[b] = (leaves[b, 0, idx].min() - margin, leaves[b, 1, idx].max() + margin,
                   bounds[idx.min()], bounds[idx.max() + 1])
    return jaws


def config5() -> Workload:
    """Double-arc VMAT on a 256x256x160 pelvis CT @ 2 mm: 2x178 control points, 80 pairs, jaws tracking
    the aperture, fluence 96x208 @ 2 mm (leaf rows misaligned with pixel rows), k = 31; the 20-iteration
    gradient-descent loop is driven by the harness."""
    rng = np.random.Generator(np.random.PCG64(1005))
    grid = centred_grid(256, 256, 160, 2.0)
    rho = pelvis_phantom(grid, rng)
    model = common_model(80, 200.0, 96, 208, 2.0, 31)
    b = np.arange(178)
    gantry = np.concatenate([(181.0 + 2.0 * b) % 360.0, (179.0 - 2.0 * b) % 360.0])
    n_cp = gantry.shape[0]
    bounds = np.asarray(model["leaf_bounds_mm"], np.float64)
    leaves, _ = _target_leaves(rng, n_cp, bounds, 0.5)
    jaws = track_jaws(leaves, bounds)
    mu = rng.uniform(1.0, 4.0, size=n_cp)
    return Workload("c5", 1005, grid, model, rho, _f32(leaves), _f32(jaws), _f32(gantry), _f32(mu),
                    backward=True, kernel_sizes=(31,), masks=pelvis_masks(grid))


# ----------------------------------------------------------------------------- small cases for tests
def tiny(seed: int = 7, nx: int = 28, ny: int = 24, nz: int = 12, spacing: float = 4.0, n_cp: int = 3,
         n_pairs: int = 6, kernel_size: int = 5, flu=(20, 16), flu_d: float = 3.0, head_scatter: bool = True,
         gantry=None, explicit_beam=None) -> Workload:
    """A few-thousand-voxel case the oracle finishes in milliseconds: random density, leaf rows misaligned
    with pixel rows, head scatter on, oblique gantry angles, several tiles and ragged tails."""
    rng = np.random.Generator(np.random.PCG64(seed))
    grid = centred_grid(nx, ny, nz, spacing)
    grid["iso"] = (1.3, -2.1, 0.7)
    rho = _f32(rng.uniform(0.2, 1.6, size=(nz, ny, nx)))
    half_v = 0.5 * flu[1] * flu_d * 0.8
    model = common_model(n_pairs, half_v, flu[0], flu[1], flu_d, kernel_size)
    if head_scatter:
        model.update(n_hs=2, hs_amp=_f32([0.04, 0.015]), hs_sigma_mm=_f32([4.0, 9.0]))
    if explicit_beam is not None:
        model.update(explicit_beam)
    half_u = 0.5 * flu[0] * flu_d
    draws = rng.uniform(-0.6 * half_u, 0.6 * half_u, size=(n_cp, 2, n_pairs))
    leaves = np.stack([draws.min(axis=1), draws.max(axis=1)], axis=1)
    jaws = np.stack([rng.uniform(-0.7 * half_u, -0.3 * half_u, n_cp), rng.uniform(0.3 * half_u, 0.7 * half_u, n_cp),
                     rng.uniform(-0.9 * half_v, -0.4 * half_v, n_cp), rng.uniform(0.4 * half_v, 0.9 * half_v, n_cp)], axis=1)
    g = rng.uniform(0.0, 360.0, size=n_cp) if gantry is None else np.asarray(gantry, np.float64)
    mu = rng.uniform(0.5, 3.0, size=n_cp)
    return Workload(f"tiny{seed}", seed, grid, model, rho, _f32(leaves), _f32(jaws), _f32(g), _f32(mu),
                    backward=True, kernel_sizes=(kernel_size,))


def seeded_dose_gradient(wl: Workload, seed: int = 0) -> np.ndarray:
    """A seeded dL/dDose field for tests that need one without running any dose engine: smooth random
    values on the workload's masks (or everywhere when it has none)."""
    rng = np.random.Generator(np.random.PCG64(10_000 + seed))
    g = rng.standard_normal((wl.grid["nz"], wl.grid["ny"], wl.grid["nx"]))
    if wl.masks:
        keep = np.zeros(g.shape, bool)
        for mask, _, _ in wl.masks.values():
            keep |= mask
        g = np.where(keep, g, 0.0)
    return _f32(g)


def objective_and_gradient(dose, masks):
    """Quadratic target/OAR objective of SURVEY.md §8(d) c4 and its dose gradient (harness code, numpy).
    L = sum_s (w_s/|s|) sum_{voxels in s} (D - p_s)^2, p_s = prescription (0 for OARs)."""
    L = 0.0
    g = np.zeros(dose.shape, np.float64)
    for mask, weight, presc in masks.values():
        n = max(int(mask.sum()), 1)
        d = dose[mask] - (presc or 0.0)
        L += weight / n * float((d * d).sum())
        g[mask] += 2.0 * weight / n * d
    return L, _f32(g)


def structure_bits(wl: Workload):
    """The workload's masks as the inputs of pdrt_objective: (uint32 [nz][ny][nx] with bit s = membership of structure s,
    lambda_s = weight_s / |s|, prescription_s), structures in the order of wl.masks."""
    shape = (wl.grid["nz"], wl.grid["ny"], wl.grid["nx"])
    bits = np.zeros(shape, np.uint32)
    lam, presc = [], []
    for s, (mask, weight, p) in enumerate(wl.masks.values()):
        bits |= mask.astype(np.uint32) << np.uint32(s)
        lam.append(weight / max(int(mask.sum()), 1))
        presc.append(p or 0.0)
    return bits, _f32(lam), _f32(presc)


def plan_limits(wl: Workload) -> dict:
    """Limits of the Eq. 1-3 projection for the planning loop (DESIGN.md §4 c5): leaf gap >= 0.5 mm, pair centres within the
    fluence map's half width, MU >= 0.1; jaws are tracked, their limits are wide open."""
    half_u = 0.5 * wl.model["flu_nu"] * wl.model["flu_du"]
    return dict(leaf_w_min=0.5, leaf_F=half_u, jaw_w_min=0.0, jaw_Fx=1e6, jaw_Fy=1e6, mu_eps=0.1)


CONFIGS = {"c1": config1, "c2": config2, "c3": config3, "c4": config4, "c5": config5}
