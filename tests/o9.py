"""Config-4 mask system (O9): harness-level composition of the split-step
propagator A, two phase masks and a 2f system, with the Gaussian-overlap loss and its gradients through
the adjoint split step.  Written twice: once on the CPU oracle's calls (fp64), once on the C-ABI calls.
Test infrastructure only; holds no kernel code.

  V1 = A(U0);  V2 = e^{i th1} V1;  V3 = F_c V2;  V4 = e^{i th2} V3;  V5 = F_c^-1 V4
  loss = 1 - |c|^2 / (P_T P_V),  c = sum conj(T) V5,  T = free-space-propagated input beam   ("overlap", config 4)
  G5 = -(2 / (P_T P_V)) [c T - (|c|^2 / P_V) V5];  G4 = F_c G5;  dl/dth2 = Im(G4 conj V4)
  loss = (1/N^2) sum |V5 - T|   ("mae": the paper's D2NN loss, "mean absolute error" between the
         processed field and the free-space result; read as the mean modulus of the complex difference, which is what
         an L1 loss on complex tensors computes);  G5 = (1/N^2) (V5 - T) / |V5 - T|  (0 where V5 = T)
  G2 = F_c^-1 (e^{-i th2} G4);  dl/dth1 = Im(G2 conj V2);  G1 = e^{-i th1} G2;  G0 = A^H G1 (+ dl/dphi_j)
"""
import numpy as np


def oracle_chain(orc, N, dx, lam, dz, u0, scr32, th1, th2, kw, aperture_radius=None, parallel=False, loss_kind="overlap"):
    """All quantities for ONE batch of fields on the oracle.  Returns a dict of float64 / complex128 arrays.
    aperture_radius: optional circular aperture applied to A(U0) and to the target; a real 0/1
    mask, so the adjoint applies it again.  parallel: issue the two independent propagations (through the screens,
    and through vacuum for the target) side by side."""
    ap = (lambda x: x) if aperture_radius is None else (lambda x: orc.aperture(N, dx, aperture_radius, x))
    legs = [lambda: orc.propagate(N, dx, lam, dz, u0, scr32, return_planes=True, **kw),
            lambda: orc.propagate(N, dx, lam, dz, u0, None, **kw)]
    if parallel:
        from tests.util import pmap
        (V1, planes), T = pmap(lambda f: f(), legs)
    else:
        (V1, planes), T = legs[0](), legs[1]()
    V1 = ap(V1)
    T = ap(T)
    V2 = orc.phase_mul(N, th1, V1)
    V3 = orc.dft2_centered(N, V2)
    V4 = orc.phase_mul(N, th2, V3)
    V5 = orc.dft2_centered(N, V4, inverse=True)
    B = V5.shape[0]
    c = np.array([np.vdot(T[b], V5[b]) for b in range(B)])
    PT = np.array([np.vdot(T[b], T[b]).real for b in range(B)])
    PV = np.array([np.vdot(V5[b], V5[b]).real for b in range(B)])
    if loss_kind == "mae":
        D = V5 - T
        mod = np.abs(D)
        loss = mod.mean(axis=(1, 2))
        G5 = np.where(mod > 0, D / np.where(mod > 0, mod, 1.0), 0.0) / (N * N)
    else:
        loss = 1.0 - np.abs(c) ** 2 / (PT * PV)
        al = -2.0 * c / (PT * PV)
        be = 2.0 * np.abs(c) ** 2 / (PT * PV * PV)
        G5 = al[:, None, None] * T + be[:, None, None] * V5
    G4 = orc.dft2_centered(N, G5)
    g_th2 = orc.phase_grad(N, G4, V4)
    G2 = orc.dft2_centered(N, orc.phase_mul(N, th2, G4, sign=-1.0), inverse=True)
    g_th1 = orc.phase_grad(N, G2, V2)
    G1 = ap(orc.phase_mul(N, th1, G2, sign=-1.0))
    G0, g_phi = orc.propagate_adjoint(N, dx, lam, dz, G1, scr32, planes=planes, **kw)
    return dict(loss=loss, V5=V5, g_th1=g_th1, g_th2=g_th2, g_phi=g_phi, G0=G0, planes=planes)


def gpu_chain(ssp, N, dx, lam, dz, u0, scr32, th1, th2, kw):
    """The same chain through the C-ABI binding (torch CUDA tensors in, torch tensors out)."""
    import torch
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    d_u0, d_scr, d_th1, d_th2 = cu(u0), cu(scr32), cu(th1), cu(th2)
    B, S, n_steps = u0.shape[0], scr32.shape[1], len(dz)
    planes = torch.empty((B, n_steps, N, N), dtype=torch.complex64, device="cuda")
    V1 = ssp.propagate(N, dx, lam, list(dz), d_u0, d_scr, planes=planes, **kw)
    T = ssp.propagate(N, dx, lam, list(dz), d_u0, None, **kw)
    V2 = ssp.phase_mul(N, dx, d_th1, V1)
    V3 = ssp.dft2_centered(N, dx, V2)
    V4 = ssp.phase_mul(N, dx, d_th2, V3)
    V5 = ssp.dft2_centered(N, dx, V4, inverse=True)
    ip = ssp.inner_products(N, dx, T, V5).cpu().numpy()        # <T, V5>, |T|^2, |V5|^2 in fp64
    c = ip[:, 0] + 1j * ip[:, 1]
    PT, PV = ip[:, 2], ip[:, 3]
    loss = 1.0 - np.abs(c) ** 2 / (PT * PV)
    al = -2.0 * c / (PT * PV)
    be = 2.0 * np.abs(c) ** 2 / (PT * PV * PV)
    G5 = ssp.lincomb(N, dx, list(al), T, list(be.astype(complex)), V5)
    G4 = ssp.dft2_centered(N, dx, G5)
    g_th2 = ssp.phase_grad(N, dx, G4, V4)
    G2 = ssp.dft2_centered(N, dx, ssp.phase_mul(N, dx, d_th2, G4, sign=-1.0), inverse=True)
    g_th1 = ssp.phase_grad(N, dx, G2, V2)
    G1 = ssp.phase_mul(N, dx, d_th1, G2, sign=-1.0)
    g_phi = torch.zeros((B, S, N, N), dtype=torch.float32, device="cuda")
    G0 = ssp.propagate_adjoint(N, dx, lam, list(dz), G1, d_scr, planes=planes, phase_grad=g_phi, **kw)
    return dict(loss=loss, V5=V5, g_th1=g_th1, g_th2=g_th2, g_phi=g_phi, G0=G0)
