"""Two-mask diffractive receiver trained through the adjoint split step (O9).

    V1 = aperture(A(U0));  V2 = e^{i th1} V1;  V3 = F_c V2;  V4 = e^{i th2} V3;  V5 = F_c^-1 V4
    loss = mean |V5 - T|,   T = aperture(A_vacuum(U0))      ("mae": the paper's mean-absolute-error loss; default)
    loss = 1 - |<T, V5>|^2 / (|T|^2 |V5|^2)                 ("overlap": BASELINE.json config 4's Gaussian-overlap loss, Q21)

A is the split-step propagation through one realisation of the screen stack per field.  Every array operation is
a call into libssp (propagation, lens transforms, mask multiplies, inner products, gradients, Adam update); this
module only sequences the calls and does the per-field scalar algebra of the loss on the host.  The gradients are
those of tests/o9.py (checked there against the CPU oracle and finite differences), plus the aperture, which is a
real 0/1 mask and therefore its own adjoint.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np
import torch

from . import api


@dataclass
class TwoMaskReceiver:
    ctx: api.Context
    N: int
    dx: float
    lam: float
    dz: list
    aperture_radius: Optional[float] = None      # metres; None = no aperture
    win_order: int = 16
    win_sigma_frac: float = 0.47
    h_kind: int = api.H_FRESNEL
    loss: str = "mae"                             # "mae" or "overlap" (config 4)
    lr: float = 0.01
    total_steps: int = 1000                       # length of the one-cycle schedule
    theta: list = field(default_factory=list)     # two fp32 [N][N] masks (constant-phase initialisation)
    _m: list = field(default_factory=list)
    _v: list = field(default_factory=list)
    t: int = 0

    def __post_init__(self):
        dev = torch.device("cuda", self.ctx.device)
        if not self.theta:
            self.theta = [torch.zeros((self.N, self.N), dtype=torch.float32, device=dev) for _ in range(2)]
        self._m = [torch.zeros_like(th) for th in self.theta]
        self._v = [torch.zeros_like(th) for th in self.theta]
        self._kw = dict(win_order=self.win_order, win_sigma_frac=self.win_sigma_frac, h_kind=self.h_kind)

    # ---- pieces -------------------------------------------------------------------------------------
    def _ap(self, u):
        return u if self.aperture_radius is None else self.ctx.aperture(self.N, self.dx, self.aperture_radius, u)

    def target(self, u0):
        """Free-space-propagated, apodised input beam."""
        return self._ap(self.ctx.propagate(self.N, self.dx, self.lam, self.dz, u0, None, **self._kw))

    def forward(self, u0, screens):
        c, N, dx = self.ctx, self.N, self.dx
        V1 = self._ap(c.propagate(N, dx, self.lam, self.dz, u0, screens, **self._kw))
        V2 = c.phase_mul(N, dx, self.theta[0], V1)
        V3 = c.dft2_centered(N, dx, V2)
        V4 = c.phase_mul(N, dx, self.theta[1], V3)
        V5 = c.dft2_centered(N, dx, V4, inverse=True)
        return V2, V4, V5

    def loss_and_grads(self, u0, screens, T=None, input_grad=False, device_loss=False):
        """Per-field losses (numpy fp64 [B]; with device_loss and the "mae" loss: the fp64 CUDA tensor, no host
        synchronisation) and d loss / d theta_1, d theta_2 per field (fp32 [B][N][N]); with input_grad also
        G0 = A^H(...) (the adjoint split step through the screen stack)."""
        c, N, dx = self.ctx, self.N, self.dx
        T = self.target(u0) if T is None else T
        V2, V4, V5 = self.forward(u0, screens)
        if self.loss == "mae":
            d_loss, G5 = c.mae_loss(N, dx, V5, T)                    # loss and dl/dV5 in one kernel, nothing on the host
            loss = d_loss if device_loss else d_loss.cpu().numpy()
        elif self.loss == "overlap":
            ip = c.inner_products(N, dx, T, V5).cpu().numpy()       # <T, V5>, |T|^2, |V5|^2 (fp64)
            cc = ip[:, 0] + 1j * ip[:, 1]
            PT, PV = ip[:, 2], ip[:, 3]
            loss = 1.0 - np.abs(cc) ** 2 / (PT * PV)
            al = -2.0 * cc / (PT * PV)
            be = 2.0 * np.abs(cc) ** 2 / (PT * PV * PV)
            G5 = c.lincomb(N, dx, list(al), T, list(be.astype(complex)), V5)
        else:
            raise ValueError(f"unknown loss {self.loss!r}")
        G4 = c.dft2_centered(N, dx, G5)
        g2 = c.phase_grad(N, dx, G4, V4)
        G2 = c.dft2_centered(N, dx, c.phase_mul(N, dx, self.theta[1], G4, sign=-1.0), inverse=True)
        g1 = c.phase_grad(N, dx, G2, V2)
        G0 = None
        if input_grad:
            G1 = self._ap(c.phase_mul(N, dx, self.theta[0], G2, sign=-1.0))
            G0 = c.propagate_adjoint(N, dx, self.lam, self.dz, G1, screens, **self._kw)
        return loss, g1, g2, G0

    def one_cycle_lr(self):
        """One-cycle schedule: cosine ramp lr/25 -> lr over the first 30 %, cosine decay to lr/2500."""
        s, n = self.t, max(self.total_steps, 2)
        up = max(1, int(0.3 * n))
        if s < up:
            return self.lr / 25 + (self.lr - self.lr / 25) * 0.5 * (1 - math.cos(math.pi * s / up))
        return self.lr / 2500 + (self.lr - self.lr / 2500) * 0.5 * (1 + math.cos(math.pi * min(1.0, (s - up) / max(1, n - up))))

    def train_step(self, u0, screens, T=None, sync=True):
        """One epoch: a batch of fresh turbulence realisations, gradients of the mean loss, one Adam step per mask.
        sync=False (mean-absolute-error loss): nothing of the epoch touches the host -- the mean loss comes back as a
        CUDA tensor to be read whenever the caller wants a progress figure."""
        dev = (not sync) and self.loss == "mae"
        loss, g1, g2, _ = self.loss_and_grads(u0, screens, T, device_loss=dev)
        lr = self.one_cycle_lr()
        self.t += 1
        for th, m, v, g in zip(self.theta, self._m, self._v, (g1, g2)):
            self.ctx.adam_update(self.N, self.dx, g, lr, self.t, m, v, th)
        return loss.mean() if dev else float(loss.mean())
