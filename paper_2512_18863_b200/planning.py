"""Call sequence of one planning iteration on the device (DESIGN.md §4 c5) — marshalling only.

Every step is a C-ABI call of include/pdrt.h that runs in the library's CUDA kernels; this module holds the raw
optimisation variables as torch CUDA tensors and calls the steps in order:

    theta^ = pdrt_validate(theta)          Eq. 1-3: w >= w_min, |c| <= F, MU >= eps
    jaws   = pdrt_track_jaws(theta^)       BASELINE.json configs[4]: jaws tracking the aperture
    D      = pdrt_dose(theta^, jaws)       Eq. 4-9
    L, g   = pdrt_objective(D)             Eq. 10 (power 1) or the quadratic objective (power 2)
    g^     = pdrt_dose_backward(theta^, jaws, g)
    g_th   = pdrt_validate_backward(theta, g^)
    theta  = pdrt_plan_step(theta, g_th)   normalised-gradient step

None of the calls synchronises, so the iteration can be captured once in a CUDA graph and replayed.
"""
from __future__ import annotations

import numpy as np

from .binding import Engine, PdrtLimits


class PlanLoop:
    def __init__(self, engine: Engine, leaves, mu, gantry_deg, limits: PdrtLimits, structure_bits, lam, presc, power: int = 2,
                 step_leaf_mm: float = 0.5, step_mu: float = 0.05, jaw_margin_mm: float = 5.0, open_gap_mm: float = 0.6):
        torch = engine.torch
        dev = engine.device
        f32 = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32)).to(dev)
        self.eng, self.limits = engine, limits
        self.leaves, self.mu, self.gantry = f32(leaves).clone(), f32(mu).clone(), f32(gantry_deg)    # raw variables theta
        n_cp = int(self.gantry.shape[0])
        self.bits = torch.as_tensor(np.ascontiguousarray(structure_bits).view(np.int32)).to(dev)
        self.lam, self.presc, self.power = np.asarray(lam, np.float32), np.asarray(presc, np.float32), int(power)
        self.step_leaf, self.step_mu, self.margin, self.open_gap = step_leaf_mm, step_mu, jaw_margin_mm, open_gap_mm
        # projected parameters, jaws, dose, objective gradient, gradients: allocated once
        self.p_leaves, self.p_mu = torch.empty_like(self.leaves), torch.empty_like(self.mu)
        self.jaws = torch.zeros((n_cp, 4), dtype=torch.float32, device=dev)
        self.p_jaws = torch.empty_like(self.jaws)                   # pdrt_validate writes the jaw pairs too (the raw jaws are the tracked ones)
        self.dose = torch.empty(engine.dose_shape, dtype=torch.float32, device=dev)
        self.g = torch.empty_like(self.dose)
        self.loss = torch.zeros(1, dtype=torch.float64, device=dev)
        self.gh = (torch.empty_like(self.leaves), torch.empty_like(self.jaws), torch.empty_like(self.mu))
        self.gr = (torch.empty_like(self.leaves), torch.empty_like(self.jaws), torch.empty_like(self.mu))
        self.iterations = 0

    def project(self):
        """theta^ and the tracked jaws of the current raw variables."""
        e = self.eng
        # the jaws are not optimisation variables here: they track the projected aperture (the jaw pairs that pdrt_validate
        # also projects are the previous iteration's and are not used)
        e.validate(self.limits, self.leaves, self.jaws, self.mu, out=(self.p_leaves, self.p_jaws, self.p_mu))
        e.track_jaws(self.p_leaves, self.margin, self.open_gap, out=self.jaws)
        return self.p_leaves, self.jaws, self.p_mu

    def forward_backward(self):
        """Dose, objective and the gradients w.r.t. the projected parameters for the current variables."""
        e = self.eng
        self.project()
        e.dose(self.p_leaves, self.jaws, self.gantry, self.p_mu, out=self.dose)
        e.objective(self.dose, self.bits, self.lam, self.presc, self.power, out=(self.loss, self.g))
        e.dose_backward(self.p_leaves, self.jaws, self.gantry, self.p_mu, self.g, out=self.gh)
        return self.gh

    def update(self):
        """Gradients w.r.t. the raw variables, then the normalised-gradient step."""
        e = self.eng
        e.validate_backward(self.limits, self.leaves, self.jaws, self.mu, *self.gh, out=self.gr)
        e.plan_step(self.step_leaf, self.step_mu, self.gr[0], self.gr[2], self.leaves, self.mu)

    def iterate(self):
        self.forward_backward()
        self.update()
        self.iterations += 1
