"""ctypes front-end of the float64 CPU oracle (oracle/pdrt_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Nothing under paper_2512_18863_b200/ imports it and it
imports nothing from there.  All arithmetic lives in the C file; this module only marshals
arrays (float32 inputs are widened exactly to float64) and resolves the documented defaults of
the beam grid (beam_nu/nw = nx/ny, du = dw = sx, centred on the isocentre;
ray step = 0.5 * min spacing).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pdrt_oracle.c")
_LIB = os.path.join(_HERE, "libpdrt_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C11, -O2, OpenMP, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-ffp-contract=off",
             "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("sx", C.c_double), ("sy", C.c_double), ("sz", C.c_double),
                ("ox", C.c_double), ("oy", C.c_double), ("oz", C.c_double),
                ("iso", C.c_double * 3)]


_DP = C.POINTER(C.c_double)


class _Model(C.Structure):
    _fields_ = [("sid", C.c_double),
                ("n_pairs", C.c_int), ("leaf_bounds", _DP),
                ("flu_nu", C.c_int), ("flu_nv", C.c_int), ("flu_du", C.c_double), ("flu_dv", C.c_double),
                ("tau", C.c_double), ("fwhm_mlc", C.c_double), ("fwhm_jaw", C.c_double),
                ("n_hs", C.c_int), ("hs_amp", _DP), ("hs_sigma", _DP),
                ("n_oar", C.c_int), ("oar_dr", C.c_double), ("oar", _DP),
                ("n_z", C.c_int), ("dz", C.c_double),
                ("kA", _DP), ("ka", _DP), ("kB", _DP), ("kb", _DP),
                ("kernel_size", C.c_int), ("cal", C.c_double),
                ("beam_nu", C.c_int), ("beam_nw", C.c_int),
                ("beam_du", C.c_double), ("beam_dw", C.c_double), ("beam_wmin", C.c_double),
                ("ray_step", C.c_double)]


def _d(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _p(a):
    return a.ctypes.data_as(_DP)


@dataclass
class Oracle:
    """Holds one (grid, density, beam model) and exposes the oracle's steps.

    `grid` and `model` are plain dicts with the field names of include/pdrt.h
    (pdrt_grid / pdrt_beam_model); see paper_2512_18863_b200/workloads.py.  The "_mm" suffix of
    those names is dropped here (everything is millimetres).
    """
    grid: dict
    model: dict
    density: np.ndarray
    _keep: list = field(default_factory=list, repr=False)
    _tables: dict = field(default_factory=dict, repr=False)

    def __post_init__(self):
        self.lib = C.CDLL(build())
        g = self.grid
        m = {(k[:-3] if k.endswith("_mm") else k): v for k, v in self.model.items()}
        self.density = np.ascontiguousarray(self.density, dtype=np.float32)
        assert self.density.shape == (g["nz"], g["ny"], g["nx"])
        # documented defaults (include/pdrt.h): beam_nu == 0 selects the default beam grid as a whole
        if not m.get("beam_nu"):
            m["beam_nu"], m["beam_nw"] = g["nx"], g["ny"]
            m["beam_du"] = m["beam_dw"] = g["sx"]
            m["beam_wmin"] = -0.5 * (m["beam_nw"] - 1) * m["beam_dw"]
        if not m.get("ray_step"):
            m["ray_step"] = 0.5 * min(g["sx"], g["sy"], g["sz"])
        self.m = m
        self.G = _Grid(g["nx"], g["ny"], g["nz"], g["sx"], g["sy"], g["sz"], g["ox"], g["oy"], g["oz"],
                       (C.c_double * 3)(*[float(v) for v in g["iso"]]))
        arr = {k: _d(m[k]) for k in ("leaf_bounds", "kA", "ka", "kB", "kb")}
        arr["hs_amp"] = _d(m.get("hs_amp", [])) if m.get("n_hs", 0) else _d([0.0])
        arr["hs_sigma"] = _d(m.get("hs_sigma", [])) if m.get("n_hs", 0) else _d([0.0])
        arr["oar"] = _d(m.get("oar", [])) if m.get("n_oar", 0) else _d([1.0])
        self._keep.append(arr)
        self.M = _Model(float(m["sid"]), int(m["n_pairs"]), _p(arr["leaf_bounds"]),
                        int(m["flu_nu"]), int(m["flu_nv"]), float(m["flu_du"]), float(m["flu_dv"]),
                        float(m["tau"]), float(m["fwhm_mlc"]), float(m["fwhm_jaw"]),
                        int(m.get("n_hs", 0)), _p(arr["hs_amp"]), _p(arr["hs_sigma"]),
                        int(m.get("n_oar", 0)), float(m.get("oar_dr", 1.0)), _p(arr["oar"]),
                        int(m["n_z"]), float(m["dz"]), _p(arr["kA"]), _p(arr["ka"]), _p(arr["kB"]), _p(arr["kb"]),
                        int(m["kernel_size"]), float(m["cal"]),
                        int(m["beam_nu"]), int(m["beam_nw"]), float(m["beam_du"]), float(m["beam_dw"]),
                        float(m["beam_wmin"]), float(m["ray_step"]))
        self.lib.orc_ov.restype = C.c_double
        self.lib.orc_dov_dhi.restype = C.c_double
        self.lib.orc_dov_dlo.restype = C.c_double
        for f in ("orc_ov", "orc_dov_dhi", "orc_dov_dlo"):
            getattr(self.lib, f).argtypes = [C.c_double] * 4
        self.lib.orc_gauss_taps.restype = C.c_int
        self.lib.orc_gauss_taps.argtypes = [C.c_double, C.c_double, _DP]
        self.lib.orc_num_threads.restype = C.c_int

    # ---- shapes
    @property
    def flu_shape(self):
        return (self.m["flu_nv"], self.m["flu_nu"])

    @property
    def beam_shape(self):
        return (self.m["beam_nw"], self.grid["nz"], self.m["beam_nu"])

    @property
    def dose_shape(self):
        return (self.grid["nz"], self.grid["ny"], self.grid["nx"])

    def set_kernel_size(self, k: int):
        self.m["kernel_size"] = int(k)
        self.M.kernel_size = int(k)

    def _w_tab(self):
        """orc_kernel_table for the current kernel size, built once per size (the table depends on nothing else)."""
        k = int(self.m["kernel_size"])
        if k not in self._tables:
            self._tables[k] = _d(self.kernel_table())
        return self._tables[k]

    def num_threads(self) -> int:
        return int(self.lib.orc_num_threads())

    # ---- scalar helpers (Eq. 4)
    def ov(self, c, D, lo, hi):
        return self.lib.orc_ov(c, D, lo, hi)

    def dov_dhi(self, c, D, lo, hi):
        return self.lib.orc_dov_dhi(c, D, lo, hi)

    def dov_dlo(self, c, D, lo, hi):
        return self.lib.orc_dov_dlo(c, D, lo, hi)

    def gauss_taps(self, sigma, D):
        g = np.zeros(129)
        T = self.lib.orc_gauss_taps(float(sigma), float(D), _p(g))
        return T, g[:2 * T + 1].copy()

    def blur_axis(self, a, axis, T, g, transpose=False):
        a = _d(a)
        out = np.zeros_like(a)
        g = _d(g)
        fn = self.lib.orc_blur_axis_T if transpose else self.lib.orc_blur_axis
        fn(_p(a), _p(out), C.c_int(a.shape[1]), C.c_int(a.shape[0]), C.c_int(axis), C.c_int(T), _p(g))
        return out

    # ---- steps
    def fluence(self, leaves, jaws, parts=False):
        lv, jw = _d(leaves), _d(jaws)
        assert lv.shape == (2, self.m["n_pairs"]) and jw.shape == (4,)
        out = np.zeros(self.flu_shape)
        if parts:
            A, J, P0 = np.zeros(self.flu_shape), np.zeros(self.flu_shape), np.zeros(self.flu_shape)
            self.lib.orc_fluence(C.byref(self.M), _p(lv), _p(jw), _p(A), _p(J), _p(P0), _p(out))
            return out, A, J, P0
        self.lib.orc_fluence(C.byref(self.M), _p(lv), _p(jw), None, None, None, _p(out))
        return out

    def fluence_adjoint(self, leaves, jaws, gPhimap):
        lv, jw, gp = _d(leaves), _d(jaws), _d(gPhimap)
        dl, dj = np.zeros((2, self.m["n_pairs"])), np.zeros(4)
        self.lib.orc_fluence_adjoint(C.byref(self.M), _p(lv), _p(jw), _p(gp), _p(dl), _p(dj))
        return dl, dj

    def radiological_depth(self, gantry_deg):
        z = np.zeros(self.m["beam_nw"])
        self.lib.orc_radiological_depth(C.byref(self.G), self.density.ctypes.data_as(C.c_void_p), C.byref(self.M),
                                        C.c_double(float(gantry_deg)), _p(z))
        return z

    def kernel_table(self):
        k = self.m["kernel_size"]
        W = np.zeros((self.m["n_z"], k, k))
        self.lib.orc_kernel_table(C.byref(self.M), C.c_double(self.grid["sz"]), _p(W))
        return W

    def slice_kernel(self, W_tab, z):
        k = self.m["kernel_size"]
        W = np.zeros((k, k))
        Wt = _d(W_tab)
        self.lib.orc_slice_kernel(C.byref(self.M), _p(Wt), C.c_double(float(z)), _p(W))
        return W

    def project(self, Phimap):
        P = _d(Phimap)
        out = np.zeros(self.beam_shape)
        self.lib.orc_project(C.byref(self.G), C.byref(self.M), _p(P), _p(out))
        return out

    def project_adjoint(self, H):
        H = _d(H)
        out = np.zeros(self.flu_shape)
        self.lib.orc_project_adjoint(C.byref(self.G), C.byref(self.M), _p(H), _p(out))
        return out

    def convolve(self, W_tab, z, Phivol, transpose=False):
        Wt, z, P = _d(W_tab), _d(z), _d(Phivol)
        out = np.zeros(self.beam_shape)
        fn = self.lib.orc_convolve_adjoint if transpose else self.lib.orc_convolve
        fn(C.byref(self.G), C.byref(self.M), _p(Wt), _p(z), _p(P), _p(out))
        return out

    def resample_add(self, gantry_deg, scale, Db, dose=None):
        Db = _d(Db)
        if dose is None:
            dose = np.zeros(self.dose_shape)
        self.lib.orc_resample_add(C.byref(self.G), C.byref(self.M), C.c_double(float(gantry_deg)),
                                  C.c_double(float(scale)), _p(Db), _p(dose))
        return dose

    def resample_adjoint(self, gantry_deg, gdose):
        g = np.ascontiguousarray(gdose, dtype=np.float32)
        out = np.zeros(self.beam_shape)
        self.lib.orc_resample_adjoint(C.byref(self.G), C.byref(self.M), C.c_double(float(gantry_deg)),
                                      g.ctypes.data_as(C.c_void_p), _p(out))
        return out

    def beam_dose(self, leaves, jaws, gantry_deg, W_tab=None):
        Wt = self._w_tab() if W_tab is None else _d(W_tab)
        lv, jw = _d(leaves), _d(jaws)
        out = np.zeros(self.beam_shape)
        self.lib.orc_beam_dose(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(Wt),
                               _p(lv), _p(jw), C.c_double(float(gantry_deg)), _p(out))
        return out

    # ---- whole path
    def _cp_args(self, leaves, jaws, gantry_deg, mu):
        lv, jw, ga, mu = _d(leaves), _d(jaws), _d(gantry_deg), _d(mu)
        n_cp = ga.shape[0]
        assert lv.shape == (n_cp, 2, self.m["n_pairs"]) and jw.shape == (n_cp, 4) and mu.shape == (n_cp,)
        return n_cp, lv, jw, ga, mu

    def dose(self, leaves, jaws, gantry_deg, mu):
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        out = np.zeros(self.dose_shape)
        self.lib.orc_dose(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()), C.c_int(n_cp),
                          _p(lv), _p(jw), _p(ga), _p(mu), _p(out))
        return out

    def dose_backward(self, leaves, jaws, gantry_deg, mu, gdose):
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        g = np.ascontiguousarray(gdose, dtype=np.float32)
        assert g.shape == self.dose_shape
        dl, dj, dm = np.zeros_like(lv), np.zeros_like(jw), np.zeros_like(mu)
        self.lib.orc_dose_backward(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p),
                                   _p(self._w_tab()), C.c_int(n_cp), _p(lv), _p(jw), _p(ga), _p(mu), g.ctypes.data_as(C.c_void_p),
                                   _p(dl), _p(dj), _p(dm))
        return dl, dj, dm

    # ---- divergent radiological depth
    @property
    def fan_shape(self):
        return (self.m["beam_nw"], self.m["flu_nv"], self.m["flu_nu"])

    def fan_depth(self, gantry_deg):
        """z_fan[k][b][a]: radiological depth (per unit axial distance) of the ray through map pixel (a,b) at slice k."""
        z = np.zeros(self.fan_shape)
        self.lib.orc_fan_depth(C.byref(self.G), self.density.ctypes.data_as(C.c_void_p), C.byref(self.M), C.c_double(float(gantry_deg)), _p(z))
        return z

    def depth_term(self, z):
        self.lib.orc_depth_term.restype = C.c_double
        return float(self.lib.orc_depth_term(C.byref(self.M), C.c_double(float(z))))

    def fan_factor(self, z_fan, z_cax):
        zf, zc = _d(z_fan), _d(z_cax)
        F = np.zeros(self.fan_shape)
        self.lib.orc_fan_factor(C.byref(self.G), C.byref(self.M), _p(zf), _p(zc), _p(F))
        return F

    def apply_fan_factor(self, F, vol):
        F, out = _d(F), _d(vol).copy()
        self.lib.orc_apply_fan_factor(C.byref(self.G), C.byref(self.M), _p(F), _p(out))
        return out

    def dose_fan(self, leaves, jaws, gantry_deg, mu):
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        out = np.zeros(self.dose_shape)
        self.lib.orc_dose_fan(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()), C.c_int(n_cp),
                              _p(lv), _p(jw), _p(ga), _p(mu), _p(out))
        return out

    def dose_backward_fan(self, leaves, jaws, gantry_deg, mu, gdose):
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        g = np.ascontiguousarray(gdose, dtype=np.float32)
        dl, dj, dm = np.zeros_like(lv), np.zeros_like(jw), np.zeros_like(mu)
        self.lib.orc_dose_backward_fan(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()),
                                       C.c_int(n_cp), _p(lv), _p(jw), _p(ga), _p(mu), g.ctypes.data_as(C.c_void_p), _p(dl), _p(dj), _p(dm))
        return dl, dj, dm

    # ---- collimator rotation
    def rotate_map(self, coll_deg, Phimap, transpose=False):
        P = _d(Phimap)
        out = np.zeros(self.flu_shape)
        fn = self.lib.orc_rotate_map_adjoint if transpose else self.lib.orc_rotate_map
        fn(C.byref(self.M), C.c_double(float(coll_deg)), _p(P), _p(out))
        return out

    def dose_coll(self, leaves, jaws, gantry_deg, coll_deg, mu):
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        co = _d(coll_deg)
        out = np.zeros(self.dose_shape)
        self.lib.orc_dose_coll(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()), C.c_int(n_cp),
                               _p(lv), _p(jw), _p(ga), _p(co), _p(mu), _p(out))
        return out

    def dose_backward_coll(self, leaves, jaws, gantry_deg, coll_deg, mu, gdose):
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        co = _d(coll_deg)
        g = np.ascontiguousarray(gdose, dtype=np.float32)
        dl, dj, dm = np.zeros_like(lv), np.zeros_like(jw), np.zeros_like(mu)
        self.lib.orc_dose_backward_coll(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()),
                                        C.c_int(n_cp), _p(lv), _p(jw), _p(ga), _p(co), _p(mu), g.ctypes.data_as(C.c_void_p), _p(dl), _p(dj), _p(dm))
        return dl, dj, dm

    def dose_fan_coll(self, leaves, jaws, gantry_deg, coll_deg, mu):
        """Divergent-depth mode and collimator rotation together (composition of the pinned steps, in the paper's order)."""
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        co = _d(coll_deg)
        out = np.zeros(self.dose_shape)
        self.lib.orc_dose_fan_coll(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()), C.c_int(n_cp),
                                   _p(lv), _p(jw), _p(ga), _p(co), _p(mu), _p(out))
        return out

    def dose_backward_fan_coll(self, leaves, jaws, gantry_deg, coll_deg, mu, gdose):
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        co = _d(coll_deg)
        g = np.ascontiguousarray(gdose, dtype=np.float32)
        dl, dj, dm = np.zeros_like(lv), np.zeros_like(jw), np.zeros_like(mu)
        self.lib.orc_dose_backward_fan_coll(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()),
                                            C.c_int(n_cp), _p(lv), _p(jw), _p(ga), _p(co), _p(mu), g.ctypes.data_as(C.c_void_p), _p(dl), _p(dj), _p(dm))
        return dl, dj, dm

    def dose_at(self, leaves, jaws, gantry_deg, mu, ijk):
        """Dose at selected voxels; ijk is [n][3] = (x index, y index, z index)."""
        n_cp, lv, jw, ga, mu = self._cp_args(leaves, jaws, gantry_deg, mu)
        ijk = np.ascontiguousarray(ijk, dtype=np.int32)
        out = np.zeros(ijk.shape[0])
        self.lib.orc_dose_at(C.byref(self.G), C.byref(self.M), self.density.ctypes.data_as(C.c_void_p), _p(self._w_tab()), C.c_int(n_cp),
                             _p(lv), _p(jw), _p(ga), _p(mu), C.c_int(ijk.shape[0]),
                             ijk.ctypes.data_as(C.c_void_p), _p(out))
        return out


# ---- planning loop: Eq. 1-3 projection, its transpose, Eq. 10 / quadratic objective,
# jaw tracking and the normalised-gradient step.  These need no grid or beam model, only the library.
def _lib():
    lib = C.CDLL(build())
    lib.orc_objective.restype = C.c_double
    lib.orc_mu_epsilon.restype = C.c_double
    lib.orc_mu_epsilon.argtypes = [C.c_double] * 3
    return lib


def plan_limits(leaf_w_min, leaf_F, jaw_w_min, jaw_Fx, jaw_Fy, mu_eps):
    """lim[6] of orc_validate: leaf w_min, leaf F, jaw w_min, jaw-x F, jaw-y F, mu_eps."""
    return _d([leaf_w_min, leaf_F, jaw_w_min, jaw_Fx, jaw_Fy, mu_eps])


def validate(lim, leaves, jaws, mu):
    lv, jw, m, lim = _d(leaves), _d(jaws), _d(mu), _d(lim)
    n_cp, _, n_pairs = lv.shape
    out = np.zeros_like(lv), np.zeros_like(jw), np.zeros_like(m)
    _lib().orc_validate(C.c_int(n_cp), C.c_int(n_pairs), _p(lim), _p(lv), _p(jw), _p(m), _p(out[0]), _p(out[1]), _p(out[2]))
    return out


def validate_adjoint(lim, leaves, jaws, mu, g_leaves_hat, g_jaws_hat, g_mu_hat):
    lv, jw, m, lim = _d(leaves), _d(jaws), _d(mu), _d(lim)
    gl, gj, gm = _d(g_leaves_hat), _d(g_jaws_hat), _d(g_mu_hat)
    n_cp, _, n_pairs = lv.shape
    out = np.zeros_like(lv), np.zeros_like(jw), np.zeros_like(m)
    _lib().orc_validate_adjoint(C.c_int(n_cp), C.c_int(n_pairs), _p(lim), _p(lv), _p(jw), _p(m), _p(gl), _p(gj), _p(gm),
                                _p(out[0]), _p(out[1]), _p(out[2]))
    return out


def mu_epsilon(dose_rate_min, delta_phi, gantry_speed_max):
    return float(_lib().orc_mu_epsilon(float(dose_rate_min), float(delta_phi), float(gantry_speed_max)))


def objective(dose, bits, lam, presc, power):
    """(L, g): weighted-sum objective (power 1 = Eq. 10, power 2 = quadratic) over structure bit masks and dL/dDose (float32)."""
    d = np.ascontiguousarray(dose, dtype=np.float32)
    b = np.ascontiguousarray(bits, dtype=np.uint32)
    lam, presc = _d(lam), _d(presc)
    g = np.zeros(d.shape, np.float32)
    L = _lib().orc_objective(C.c_size_t(d.size), d.ctypes.data_as(C.c_void_p), b.ctypes.data_as(C.c_void_p), C.c_int(len(lam)),
                             _p(lam), _p(presc), C.c_int(int(power)), g.ctypes.data_as(C.c_void_p))
    return float(L), g


def track_jaws(leaf_bounds, leaves, margin, open_gap):
    lv, lb = _d(leaves), _d(leaf_bounds)
    n_cp, _, n_pairs = lv.shape
    jaws = np.zeros((n_cp, 4))
    _lib().orc_track_jaws(C.c_int(n_cp), C.c_int(n_pairs), _p(lb), _p(lv), C.c_double(float(margin)), C.c_double(float(open_gap)), _p(jaws))
    return jaws


def plan_step(step_leaf, step_mu, g_leaves, g_mu, leaves, mu):
    """Returns the updated (leaves, mu); inputs are not modified."""
    lv, m, gl, gm = _d(leaves).copy(), _d(mu).copy(), _d(g_leaves), _d(g_mu)
    n_cp, _, n_pairs = lv.shape
    _lib().orc_plan_step(C.c_int(n_cp), C.c_int(n_pairs), C.c_double(float(step_leaf)), C.c_double(float(step_mu)), _p(gl), _p(gm), _p(lv), _p(m))
    return lv, m
