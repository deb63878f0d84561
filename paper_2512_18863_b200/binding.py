"""Thin Python binding of the C ABI in include/pdrt.h — argument marshalling only.

Every step of the dose path runs in the CUDA kernels of libpdrt.so; this module passes pointers of
torch CUDA tensors (device memory and streams are PyTorch's) or of pinned/pageable host arrays.
There is no CPU path: without the built library or without a CUDA device it raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpdrt.so")

SYMBOLS = ("pdrt_create", "pdrt_destroy", "pdrt_last_error", "pdrt_set_kernel_size", "pdrt_get_info", "pdrt_get_work",
           "pdrt_set_profiling", "pdrt_get_stage_ms", "pdrt_set_depth_mode", "pdrt_stage_fan_factor", "pdrt_set_collimator",
           "pdrt_dose", "pdrt_dose_backward", "pdrt_dose_host", "pdrt_dose_backward_host", "pdrt_dose_host_async", "pdrt_host_wait",
           "pdrt_stage_fluence", "pdrt_stage_depth", "pdrt_stage_beam_dose", "pdrt_stage_grad_fluence",
           "pdrt_mu_epsilon", "pdrt_validate", "pdrt_validate_backward", "pdrt_objective", "pdrt_objective_noalloc", "pdrt_track_jaws",
           "pdrt_plan_step")

STAGES = ("fluence", "depth", "scan", "conv", "gather", "resample_adj", "conv_adj", "project_adj", "fluence_adj", "project", "transpose")

_FP = C.POINTER(C.c_float)


class PdrtGrid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("sx", C.c_float), ("sy", C.c_float), ("sz", C.c_float),
                ("ox", C.c_float), ("oy", C.c_float), ("oz", C.c_float),
                ("iso", C.c_float * 3)]


class PdrtBeamModel(C.Structure):
    _fields_ = [("sid_mm", C.c_float),
                ("n_pairs", C.c_int32), ("leaf_bounds_mm", _FP),
                ("flu_nu", C.c_int32), ("flu_nv", C.c_int32), ("flu_du", C.c_float), ("flu_dv", C.c_float),
                ("tau", C.c_float), ("fwhm_mlc_mm", C.c_float), ("fwhm_jaw_mm", C.c_float),
                ("n_hs", C.c_int32), ("hs_amp", _FP), ("hs_sigma_mm", _FP),
                ("n_oar", C.c_int32), ("oar_dr_mm", C.c_float), ("oar", _FP),
                ("n_z", C.c_int32), ("dz_mm", C.c_float),
                ("kA", _FP), ("ka", _FP), ("kB", _FP), ("kb", _FP),
                ("kernel_size", C.c_int32), ("cal", C.c_float),
                ("beam_nu", C.c_int32), ("beam_nw", C.c_int32),
                ("beam_du", C.c_float), ("beam_dw", C.c_float), ("beam_wmin", C.c_float),
                ("ray_step_mm", C.c_float), ("depth_mode", C.c_int32)]


class PdrtInfo(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("beam_nu", C.c_int32), ("beam_nv", C.c_int32), ("beam_nw", C.c_int32),
                ("beam_du", C.c_float), ("beam_dv", C.c_float), ("beam_dw", C.c_float), ("beam_wmin", C.c_float),
                ("flu_nu", C.c_int32), ("flu_nv", C.c_int32), ("n_pairs", C.c_int32),
                ("kernel_size", C.c_int32), ("kernel_size_compiled", C.c_int32),
                ("ray_step_mm", C.c_float), ("ray_samples", C.c_int32), ("sm_count", C.c_int32),
                ("scratch_bytes", C.c_uint64), ("kernel_passes", C.c_int32)]


class PdrtWork(C.Structure):
    _fields_ = [("n_cp", C.c_int32), ("conv_items", C.c_int64), ("support_voxels", C.c_int64),
                ("footprint_voxels", C.c_int64), ("region_voxels", C.c_int64), ("conv_macs", C.c_int64),
                ("kernel_size", C.c_int32), ("kernel_size_compiled", C.c_int32),
                ("fan_rays", C.c_int64), ("ray_samples", C.c_int32), ("conv_symmetric", C.c_int32)]


class PdrtLimits(C.Structure):
    _fields_ = [("leaf_w_min", C.c_float), ("leaf_F", C.c_float), ("jaw_w_min", C.c_float),
                ("jaw_Fx", C.c_float), ("jaw_Fy", C.c_float), ("mu_eps", C.c_float)]


class PdrtError(RuntimeError):
    def __init__(self, code, message):
        super().__init__(f"pdrt error {code}: {message}")
        self.code = code


_lib = None


def load_library(path: str = LIB_PATH) -> C.CDLL:
    """Loads libpdrt.so and declares the prototypes.  Fails loudly when the CUDA extension is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: build it with `python -m paper_2512_18863_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i32 = C.c_void_p, C.c_int32
    lib.pdrt_create.argtypes = [C.POINTER(PdrtGrid), vp, C.POINTER(PdrtBeamModel), C.POINTER(vp)]
    lib.pdrt_destroy.argtypes = [vp]
    lib.pdrt_destroy.restype = None
    lib.pdrt_last_error.argtypes = [vp]
    lib.pdrt_last_error.restype = C.c_char_p
    lib.pdrt_set_kernel_size.argtypes = [vp, i32]
    lib.pdrt_set_depth_mode.argtypes = [vp, i32]
    lib.pdrt_set_collimator.argtypes = [vp, i32, vp, vp]
    lib.pdrt_stage_fan_factor.argtypes = [vp, i32, vp, vp, vp, vp, vp]
    lib.pdrt_get_info.argtypes = [vp, C.POINTER(PdrtInfo)]
    lib.pdrt_get_work.argtypes = [vp, C.POINTER(PdrtWork)]
    lib.pdrt_set_profiling.argtypes = [vp, i32]
    lib.pdrt_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i32)]
    lib.pdrt_dose.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    lib.pdrt_dose_backward.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.pdrt_dose_host.argtypes = lib.pdrt_dose.argtypes
    lib.pdrt_dose_host_async.argtypes = lib.pdrt_dose.argtypes
    lib.pdrt_host_wait.argtypes = [vp]
    lib.pdrt_dose_backward_host.argtypes = lib.pdrt_dose_backward.argtypes
    lib.pdrt_stage_fluence.argtypes = [vp, i32, vp, vp, vp, vp]
    lib.pdrt_stage_depth.argtypes = [vp, i32, vp, vp, vp]
    lib.pdrt_stage_beam_dose.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.pdrt_stage_grad_fluence.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    f32 = C.c_float
    lib.pdrt_mu_epsilon.argtypes = [f32, f32, f32]
    lib.pdrt_mu_epsilon.restype = f32
    lib.pdrt_validate.argtypes = [vp, i32, C.POINTER(PdrtLimits), vp, vp, vp, vp, vp, vp, vp]
    lib.pdrt_validate_backward.argtypes = [vp, i32, C.POINTER(PdrtLimits), vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.pdrt_objective.argtypes = [vp, vp, vp, i32, _FP, _FP, i32, vp, vp, vp]
    lib.pdrt_objective_noalloc.argtypes = lib.pdrt_objective.argtypes
    lib.pdrt_track_jaws.argtypes = [vp, i32, vp, f32, f32, vp, vp]
    lib.pdrt_plan_step.argtypes = [vp, i32, f32, f32, vp, vp, vp, vp, vp]
    for name in SYMBOLS:
        if name not in ("pdrt_destroy", "pdrt_last_error", "pdrt_mu_epsilon"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def _fp(a):
    return a.ctypes.data_as(_FP)


class Engine:
    """pdrt_engine handle.  Device tensors are torch.float32 CUDA tensors; names follow include/pdrt.h."""

    def __init__(self, grid: dict, model: dict, density, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("pdrt needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self._keep = {k: _f32(model[k]) for k in ("leaf_bounds_mm", "kA", "ka", "kB", "kb")}
        n_hs, n_oar = int(model.get("n_hs", 0)), int(model.get("n_oar", 0))
        self._keep["hs_amp"] = _f32(model["hs_amp"]) if n_hs else _f32([0])
        self._keep["hs_sigma_mm"] = _f32(model["hs_sigma_mm"]) if n_hs else _f32([0])
        self._keep["oar"] = _f32(model["oar"]) if n_oar else _f32([1])
        k = self._keep
        g = PdrtGrid(grid["nx"], grid["ny"], grid["nz"], grid["sx"], grid["sy"], grid["sz"],
                     grid["ox"], grid["oy"], grid["oz"], (C.c_float * 3)(*[float(v) for v in grid["iso"]]))
        m = PdrtBeamModel(model["sid_mm"], model["n_pairs"], _fp(k["leaf_bounds_mm"]),
                          model["flu_nu"], model["flu_nv"], model["flu_du"], model["flu_dv"],
                          model["tau"], model["fwhm_mlc_mm"], model["fwhm_jaw_mm"],
                          n_hs, _fp(k["hs_amp"]), _fp(k["hs_sigma_mm"]),
                          n_oar, float(model.get("oar_dr_mm", 1.0)), _fp(k["oar"]),
                          model["n_z"], model["dz_mm"], _fp(k["kA"]), _fp(k["ka"]), _fp(k["kB"]), _fp(k["kb"]),
                          model["kernel_size"], model["cal"],
                          int(model.get("beam_nu", 0)), int(model.get("beam_nw", 0)),
                          float(model.get("beam_du", 0.0)), float(model.get("beam_dw", 0.0)),
                          float(model.get("beam_wmin", 0.0)), float(model.get("ray_step_mm", 0.0)), int(model.get("depth_mode", 0)))
        if isinstance(density, torch.Tensor):
            dens = density.to(dtype=torch.float32).contiguous()
            dptr = dens.data_ptr()
        else:
            dens = _f32(density)
            dptr = dens.ctypes.data
        assert tuple(dens.shape) == (grid["nz"], grid["ny"], grid["nx"])
        handle = C.c_void_p()
        rc = self.lib.pdrt_create(C.byref(g), C.c_void_p(dptr), C.byref(m), C.byref(handle))
        if rc != 0:
            raise PdrtError(rc, self.lib.pdrt_last_error(None).decode())
        self.handle = handle
        self.n_pairs = int(model["n_pairs"])
        self.info = self.get_info()

    # ---- housekeeping
    def close(self):
        if getattr(self, "handle", None):
            self.lib.pdrt_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise PdrtError(rc, self.lib.pdrt_last_error(self.handle).decode())

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def _dev(self, t, shape=None):
        torch = self.torch
        if not isinstance(t, torch.Tensor):
            t = torch.as_tensor(np.asarray(t, dtype=np.float32))
        t = t.to(device=self.device, dtype=torch.float32).contiguous()
        if shape is not None:
            assert tuple(t.shape) == tuple(shape), (tuple(t.shape), tuple(shape))
        return t

    def get_info(self) -> PdrtInfo:
        info = PdrtInfo()
        self._check(self.lib.pdrt_get_info(self.handle, C.byref(info)))
        return info

    def get_work(self) -> PdrtWork:
        w = PdrtWork()
        self._check(self.lib.pdrt_get_work(self.handle, C.byref(w)))
        return w

    def set_profiling(self, enable: bool):
        self._check(self.lib.pdrt_set_profiling(self.handle, int(bool(enable))))

    def get_stage_ms(self):
        """(ms, launches) per stage of the most recent call, as dicts keyed by STAGES; synchronises."""
        ms = (C.c_float * len(STAGES))()
        n = (C.c_int32 * len(STAGES))()
        self._check(self.lib.pdrt_get_stage_ms(self.handle, ms, n))
        return dict(zip(STAGES, [float(v) for v in ms])), dict(zip(STAGES, [int(v) for v in n]))

    def set_kernel_size(self, k: int):
        self._check(self.lib.pdrt_set_kernel_size(self.handle, int(k)))
        self.info = self.get_info()

    def set_depth_mode(self, mode: int):
        """0 = central-axis ray (the paper's mode), 1 = one diverging ray per fluence-map pixel (PDRT_DEPTH_FAN)."""
        self._check(self.lib.pdrt_set_depth_mode(self.handle, int(mode)))

    def set_collimator(self, coll_deg):
        """Per-control-point collimator angles [n_cp] for subsequent calls (None removes them)."""
        if coll_deg is None:
            self._check(self.lib.pdrt_set_collimator(self.handle, 0, None, self._stream()))
            return
        co = self._dev(coll_deg)
        self._check(self.lib.pdrt_set_collimator(self.handle, int(co.shape[0]), co.data_ptr(), self._stream()))

    def stage_fan_factor(self, leaves, jaws, gantry_deg):
        ga = self._dev(gantry_deg)
        n_cp = int(ga.shape[0])
        lv, jw = self._dev(leaves, (n_cp, 2, self.n_pairs)), self._dev(jaws, (n_cp, 4))
        out = self.torch.empty((n_cp, self.info.beam_nw, *self.flu_shape), dtype=self.torch.float32, device=self.device)
        self._check(self.lib.pdrt_stage_fan_factor(self.handle, n_cp, lv.data_ptr(), jw.data_ptr(), ga.data_ptr(), out.data_ptr(), self._stream()))
        return out

    @property
    def dose_shape(self):
        return (self.info.nz, self.info.ny, self.info.nx)

    @property
    def beam_shape(self):
        return (self.info.beam_nw, self.info.beam_nv, self.info.beam_nu)

    @property
    def flu_shape(self):
        return (self.info.flu_nv, self.info.flu_nu)

    def _params(self, leaves, jaws, gantry_deg, mu):
        gantry_deg = self._dev(gantry_deg)
        n_cp = int(gantry_deg.shape[0])
        return (n_cp, self._dev(leaves, (n_cp, 2, self.n_pairs)), self._dev(jaws, (n_cp, 4)), gantry_deg,
                self._dev(mu, (n_cp,)))

    # ---- the three calls of the boundary
    def dose(self, leaves, jaws, gantry_deg, mu, out=None):
        """pdrt_dose: device tensors in, dose [nz][ny][nx] out (asynchronous on the current stream)."""
        n_cp, lv, jw, ga, mu = self._params(leaves, jaws, gantry_deg, mu)
        if out is None:
            out = self.torch.empty(self.dose_shape, dtype=self.torch.float32, device=self.device)
        self._check(self.lib.pdrt_dose(self.handle, n_cp, lv.data_ptr(), jw.data_ptr(), ga.data_ptr(), mu.data_ptr(),
                                       out.data_ptr(), self._stream()))
        return out

    def dose_backward(self, leaves, jaws, gantry_deg, mu, dL_ddose, out=None):
        """pdrt_dose_backward: returns (d_leaves, d_jaws, d_mu)."""
        torch = self.torch
        n_cp, lv, jw, ga, mu = self._params(leaves, jaws, gantry_deg, mu)
        g = self._dev(dL_ddose, self.dose_shape)
        if out is None:
            out = (torch.empty_like(lv), torch.empty_like(jw), torch.empty_like(mu))
        dl, dj, dm = out
        self._check(self.lib.pdrt_dose_backward(self.handle, n_cp, lv.data_ptr(), jw.data_ptr(), ga.data_ptr(),
                                                mu.data_ptr(), g.data_ptr(), dl.data_ptr(), dj.data_ptr(),
                                                dm.data_ptr(), self._stream()))
        return dl, dj, dm

    # ---- planning-loop steps (device tensors; asynchronous on the current stream)
    def validate(self, limits: PdrtLimits, leaves, jaws, mu, out=None):
        """pdrt_validate (Eq. 1-3): returns the projected (leaves, jaws, mu)."""
        torch = self.torch
        jw = self._dev(jaws)
        n_cp = int(jw.shape[0])
        lv, mu = self._dev(leaves, (n_cp, 2, self.n_pairs)), self._dev(mu, (n_cp,))
        if out is None:
            out = (torch.empty_like(lv), torch.empty_like(jw), torch.empty_like(mu))
        self._check(self.lib.pdrt_validate(self.handle, n_cp, C.byref(limits), lv.data_ptr(), jw.data_ptr(), mu.data_ptr(),
                                           out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), self._stream()))
        return out

    def validate_backward(self, limits: PdrtLimits, leaves, jaws, mu, g_leaves_hat, g_jaws_hat, g_mu_hat, out=None):
        """pdrt_validate_backward: gradients w.r.t. the raw parameters from gradients w.r.t. the projected ones."""
        torch = self.torch
        jw = self._dev(jaws)
        n_cp = int(jw.shape[0])
        lv, mu = self._dev(leaves, (n_cp, 2, self.n_pairs)), self._dev(mu, (n_cp,))
        gl, gj, gm = self._dev(g_leaves_hat, lv.shape), self._dev(g_jaws_hat, jw.shape), self._dev(g_mu_hat, mu.shape)
        if out is None:
            out = (torch.empty_like(lv), torch.empty_like(jw), torch.empty_like(mu))
        self._check(self.lib.pdrt_validate_backward(self.handle, n_cp, C.byref(limits), lv.data_ptr(), jw.data_ptr(), mu.data_ptr(),
                                                    gl.data_ptr(), gj.data_ptr(), gm.data_ptr(),
                                                    out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), self._stream()))
        return out

    def mu_epsilon(self, dose_rate_min, delta_phi_deg, gantry_speed_max) -> float:
        return float(self.lib.pdrt_mu_epsilon(dose_rate_min, delta_phi_deg, gantry_speed_max))

    def objective(self, dose, structure_bits, lam, presc, power, out=None):
        """pdrt_objective: returns (loss as a 1-element float64 device tensor, dL/dDose)."""
        torch = self.torch
        d = self._dev(dose, self.dose_shape)
        assert structure_bits.dtype == torch.int32 and structure_bits.is_cuda and structure_bits.is_contiguous()   # uint32 bit patterns
        assert tuple(structure_bits.shape) == self.dose_shape
        lam, presc = _f32(lam), _f32(presc)
        if out is None:
            out = (torch.empty(1, dtype=torch.float64, device=self.device), torch.empty_like(d))
        loss, g = out
        self._check(self.lib.pdrt_objective(self.handle, d.data_ptr(), structure_bits.data_ptr(), len(lam), _fp(lam), _fp(presc),
                                            int(power), g.data_ptr(), loss.data_ptr(), self._stream()))
        return loss, g

    def objective_noalloc(self, dose, structure_bits, lam, presc, power, out):
        """pdrt_objective_noalloc: pdrt_objective on the library's static device scratch — no device allocation in the call, so
        `out` = (loss: 1-element float64 device tensor, dL/dDose: float32 device tensor of the dose shape) and a device-resident
        float32 `dose` are the caller's.  Calls on one GPU share the scratch and must not overlap."""
        torch = self.torch
        loss, g = out
        for t, dt in ((dose, torch.float32), (g, torch.float32), (structure_bits, torch.int32)):
            assert t.is_cuda and t.is_contiguous() and t.dtype == dt and tuple(t.shape) == self.dose_shape
        assert loss.is_cuda and loss.dtype == torch.float64 and loss.numel() == 1
        lam, presc = _f32(lam), _f32(presc)
        self._check(self.lib.pdrt_objective_noalloc(self.handle, dose.data_ptr(), structure_bits.data_ptr(), len(lam), _fp(lam), _fp(presc),
                                                    int(power), g.data_ptr(), loss.data_ptr(), self._stream()))
        return loss, g

    def track_jaws(self, leaves, margin_mm, open_gap_mm, out=None):
        lv = self._dev(leaves)
        n_cp = int(lv.shape[0])
        if out is None:
            out = self.torch.empty((n_cp, 4), dtype=self.torch.float32, device=self.device)
        self._check(self.lib.pdrt_track_jaws(self.handle, n_cp, lv.data_ptr(), margin_mm, open_gap_mm, out.data_ptr(), self._stream()))
        return out

    def plan_step(self, step_leaf_mm, step_mu, g_leaves, g_mu, leaves, mu):
        """pdrt_plan_step: updates `leaves` and `mu` (float32 CUDA tensors) in place."""
        torch = self.torch
        for t in (g_leaves, g_mu, leaves, mu):
            assert isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
        n_cp = int(mu.shape[0])
        self._check(self.lib.pdrt_plan_step(self.handle, n_cp, step_leaf_mm, step_mu, g_leaves.data_ptr(), g_mu.data_ptr(),
                                            leaves.data_ptr(), mu.data_ptr(), self._stream()))
        return leaves, mu

    # ---- host-buffer variants (copies inside the call; synchronous)
    def dose_host(self, leaves, jaws, gantry_deg, mu, out):
        """pdrt_dose_host: CPU tensors / arrays in (pinned for speed), dose written into `out` (CPU)."""
        n_cp = int(gantry_deg.shape[0])
        self._check(self.lib.pdrt_dose_host(self.handle, n_cp, _hptr(leaves), _hptr(jaws), _hptr(gantry_deg), _hptr(mu),
                                            _hptr(out), self._stream()))
        return out

    def dose_host_async(self, leaves, jaws, gantry_deg, mu, out):
        """pdrt_dose_host_async: as dose_host, but returns while the dose is still on its way to `out` (pinned); see host_wait."""
        n_cp = int(gantry_deg.shape[0])
        self._check(self.lib.pdrt_dose_host_async(self.handle, n_cp, _hptr(leaves), _hptr(jaws), _hptr(gantry_deg), _hptr(mu),
                                                  _hptr(out), self._stream()))
        return out

    def host_wait(self):
        self._check(self.lib.pdrt_host_wait(self.handle))

    def dose_backward_host(self, leaves, jaws, gantry_deg, mu, dL_ddose, d_leaves, d_jaws, d_mu):
        n_cp = int(gantry_deg.shape[0])
        self._check(self.lib.pdrt_dose_backward_host(self.handle, n_cp, _hptr(leaves), _hptr(jaws), _hptr(gantry_deg),
                                                     _hptr(mu), _hptr(dL_ddose), _hptr(d_leaves), _hptr(d_jaws),
                                                     _hptr(d_mu), self._stream()))
        return d_leaves, d_jaws, d_mu

    # ---- stage taps (parity tests)
    def stage_fluence(self, leaves, jaws):
        jw = self._dev(jaws)
        n_cp = int(jw.shape[0])
        lv = self._dev(leaves, (n_cp, 2, self.n_pairs))
        out = self.torch.empty((n_cp, *self.flu_shape), dtype=self.torch.float32, device=self.device)
        self._check(self.lib.pdrt_stage_fluence(self.handle, n_cp, lv.data_ptr(), jw.data_ptr(), out.data_ptr(), self._stream()))
        return out

    def stage_depth(self, gantry_deg):
        ga = self._dev(gantry_deg)
        out = self.torch.empty((int(ga.shape[0]), self.info.beam_nw), dtype=self.torch.float32, device=self.device)
        self._check(self.lib.pdrt_stage_depth(self.handle, int(ga.shape[0]), ga.data_ptr(), out.data_ptr(), self._stream()))
        return out

    def stage_beam_dose(self, leaves, jaws, gantry_deg):
        lv, jw, ga = self._dev(leaves, (1, 2, self.n_pairs)), self._dev(jaws, (1, 4)), self._dev(gantry_deg, (1,))
        out = self.torch.empty(self.beam_shape, dtype=self.torch.float32, device=self.device)
        self._check(self.lib.pdrt_stage_beam_dose(self.handle, lv.data_ptr(), jw.data_ptr(), ga.data_ptr(), out.data_ptr(), self._stream()))
        return out

    def stage_grad_fluence(self, leaves, jaws, gantry_deg, dL_ddose):
        ga = self._dev(gantry_deg)
        n_cp = int(ga.shape[0])
        lv, jw = self._dev(leaves, (n_cp, 2, self.n_pairs)), self._dev(jaws, (n_cp, 4))
        g = self._dev(dL_ddose, self.dose_shape)
        out = self.torch.empty((n_cp, *self.flu_shape), dtype=self.torch.float32, device=self.device)
        self._check(self.lib.pdrt_stage_grad_fluence(self.handle, n_cp, lv.data_ptr(), jw.data_ptr(), ga.data_ptr(),
                                                     g.data_ptr(), out.data_ptr(), self._stream()))
        return out


def _hptr(a):
    """Host pointer of a contiguous float32 CPU torch tensor or numpy array."""
    if hasattr(a, "data_ptr"):
        assert a.device.type == "cpu" and a.is_contiguous() and a.element_size() == 4
        return C.c_void_p(a.data_ptr())
    assert isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous
    return C.c_void_p(a.ctypes.data)
