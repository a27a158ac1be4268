"""Seeded synthetic inputs and workload descriptors (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path's tests/bench and the CPU oracle, and so it
holds none of the method's arithmetic: only random draws, the input beams and the
numbers that describe each workload.  Recipe:

  noise for realisation b of config c:  rng = default_rng([c, seed, b])
     draw order: high-frequency  standard_normal(float32) [S][N][N][2]
                 then subharmonic standard_normal(float32) [S][Np][3][3][2]
                 then, for temporal workloads, the same pair again per time step.
  beams: collimated Gaussian U0 = exp(-r^2/w0^2) or plane wave U0 = 1.
  masks (config 4): uniform [0, 2 pi) from default_rng([4, seed, 1000 + m]).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

PSD_KOLMOGOROV, PSD_VON_KARMAN, PSD_OCEAN_NIKISHOV, PSD_POWER_LAW = 0, 1, 2, 3


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config.  Lengths in metres."""
    cid: int
    name: str
    N: int
    dx: float
    lam: float
    L: float
    S: int                      # screens = split steps (equally spaced, dz = L/S; Q11)
    B: int                      # realisations in the full config
    psd_kind: int
    cn2: float = 0.0
    L0: float = 0.0
    l0: float = 0.0
    n_sh: int = 0
    beam: str = "gaussian"      # or "plane"
    w0: float = 0.0
    win_order: int = 16         # super-Gaussian absorbing window (Q12)
    win_sigma_frac: float = 0.47
    ar_a: float = 0.0           # AR coefficient (config 3)
    T_steps: int = 0            # time steps (config 3)
    chi_T: float = 0.0          # ocean
    eps: float = 0.0
    w: float = 0.0
    cn2_sweep: tuple = ()

    @property
    def dz(self) -> np.ndarray:
        return np.full(self.S, self.L / self.S, dtype=np.float64)

    @property
    def cn2_list(self) -> np.ndarray:
        return np.full(self.S, self.cn2, dtype=np.float64)

    def psd_dict(self) -> dict:
        return dict(kind=self.psd_kind, L0=self.L0, l0=self.l0, km_coeff=0.0,
                    chi_T=self.chi_T, eps=self.eps, w=self.w, eta=0.0)


CONFIGS = {
    1: Workload(1, "cfg1_gaussian_vk_128", N=128, dx=1e-3, lam=1.55e-6, L=1000.0, S=5, B=4,
                psd_kind=PSD_VON_KARMAN, cn2=1e-14, L0=10.0, l0=5e-3, n_sh=3,
                beam="gaussian", w0=2e-2),
    2: Workload(2, "cfg2_plane_kolmogorov_512", N=512, dx=2e-3, lam=1.064e-6, L=2000.0, S=10, B=64,
                psd_kind=PSD_KOLMOGOROV, cn2=1e-15, n_sh=0, beam="plane",
                cn2_sweep=(1e-15, 1e-14, 1e-13)),
    3: Workload(3, "cfg3_temporal_vk_1024", N=1024, dx=1e-3, lam=1.55e-6, L=3000.0, S=20, B=32,
                psd_kind=PSD_VON_KARMAN, cn2=5e-15, L0=20.0, l0=2e-3, n_sh=3,
                beam="gaussian", w0=3e-2, ar_a=0.99, T_steps=100),
    4: Workload(4, "cfg4_adjoint_2048", N=2048, dx=0.5e-3, lam=0.85e-6, L=1500.0, S=30, B=8,
                psd_kind=PSD_KOLMOGOROV, cn2=1e-13, n_sh=0, beam="gaussian", w0=4e-2),
    5: Workload(5, "cfg5_ocean_4096", N=4096, dx=0.25e-3, lam=0.532e-6, L=50.0, S=20, B=2,
                psd_kind=PSD_OCEAN_NIKISHOV, n_sh=4, beam="gaussian", w0=5e-3,
                chi_T=1e-7, eps=1e-5, w=-2.0),
}


def noise(cid: int, seed: int, b: int, S: int, N: int, n_sh: int, frames: int = 1):
    """Host white noise for ONE realisation b.

    Returns a list of `frames` pairs (hi, sh): hi float32 [S][N][N][2],
    sh float32 [S][max(n_sh,1)][3][3][2] (all zeros' worth of draws skipped when n_sh == 0).
    Frame 0 seeds the screens; frames 1.. are the fresh noise of successive AR steps.
    """
    rng = np.random.default_rng([cid, seed, b])
    out = []
    for _ in range(frames):
        hi = rng.standard_normal((S, N, N, 2), dtype=np.float32)
        sh = (rng.standard_normal((S, n_sh, 3, 3, 2), dtype=np.float32)
              if n_sh > 0 else np.zeros((S, 1, 3, 3, 2), dtype=np.float32))
        out.append((hi, sh))
    return out


def noise_batch(cid: int, seed: int, B: int, S: int, N: int, n_sh: int, frame: int = 0, b0: int = 0):
    """Stacked noise of realisations b0..b0+B-1 at one frame: ([B][S][N][N][2], [B][S][Np][3][3][2])."""
    his, shs = [], []
    for b in range(b0, b0 + B):
        fr = noise(cid, seed, b, S, N, n_sh, frames=frame + 1)[frame]
        his.append(fr[0])
        shs.append(fr[1])
    return np.stack(his), np.stack(shs)


def coords(N: int, dx: float) -> np.ndarray:
    return (np.arange(N) - N // 2) * dx


def gaussian_beam(N: int, dx: float, w0: float, B: int = 1) -> np.ndarray:
    """Collimated Gaussian input field U0 = exp(-r^2/w0^2), complex64 [B][N][N]."""
    x = coords(N, dx)
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    u = np.exp(-r2 / (w0 * w0)).astype(np.complex64)
    return np.broadcast_to(u, (B, N, N)).copy()


def plane_wave(N: int, B: int = 1) -> np.ndarray:
    return np.ones((B, N, N), dtype=np.complex64)


def input_field(wl: Workload, B: Optional[int] = None) -> np.ndarray:
    B = wl.B if B is None else B
    return plane_wave(wl.N, B) if wl.beam == "plane" else gaussian_beam(wl.N, wl.dx, wl.w0, B)


def random_field(N: int, B: int, seed: int) -> np.ndarray:
    """Unstructured complex64 test field (adjoint-identity and parity tests)."""
    rng = np.random.default_rng([99, seed])
    return (rng.standard_normal((B, N, N), dtype=np.float32)
            + 1j * rng.standard_normal((B, N, N), dtype=np.float32)).astype(np.complex64)


def random_screens(N: int, B: int, S: int, seed: int, rms: float = 1.5) -> np.ndarray:
    """Smooth-ish random phase maps in radians, float32 [B][S][N][N], for propagator-only tests.

    Box-blurred white noise plus a tilt: only a stand-in input with the magnitude range of
    real screens (a few to tens of radians); it is not the method's screen generator."""
    rng = np.random.default_rng([98, seed])
    w = rng.standard_normal((B, S, N, N)).astype(np.float64)
    for ax in (2, 3):
        w = (w + np.roll(w, 1, ax) + np.roll(w, -1, ax) + np.roll(w, 2, ax) + np.roll(w, -2, ax)) / 5.0
    w *= rms / w.std()
    x = np.arange(N) - N // 2
    tilt = rng.standard_normal((B, S, 2))
    w += (tilt[..., 0, None, None] * x[None, None, None, :]
          + tilt[..., 1, None, None] * x[None, None, :, None]) * (8.0 / N)
    return w.astype(np.float32)


def phase_masks(seed: int, N: int, n_masks: int = 2) -> np.ndarray:
    """Config 4: uniform-random phase masks in [0, 2 pi), float32 [n_masks][N][N]."""
    out = []
    for m in range(n_masks):
        rng = np.random.default_rng([4, seed, 1000 + m])
        out.append((rng.random((N, N), dtype=np.float32) * np.float32(2 * np.pi)).astype(np.float32))
    return np.stack(out)
