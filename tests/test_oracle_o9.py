"""Pin of the config-4 mask-system composition (tests/o9.py, O9) on the CPU oracle: every gradient
the chain returns equals a central finite difference of the loss (P8 extended to the whole system)."""
import numpy as np
import pytest

from paper_2604_07248_b200 import synth
from tests import o9


def _loss(orc, N, dx, lam, dz, u0, scr, th1, th2, kw, R=None, kind="overlap"):
    ap = (lambda x: x) if R is None else (lambda x: orc.aperture(N, dx, R, x))
    V1 = ap(orc.propagate(N, dx, lam, dz, u0, scr, **kw))
    T = ap(orc.propagate(N, dx, lam, dz, u0, None, **kw))
    V5 = orc.dft2_centered(N, orc.phase_mul(N, th2, orc.dft2_centered(N, orc.phase_mul(N, th1, V1))), inverse=True)
    if kind == "mae":                                            # mean absolute error against the free-space field
        return np.mean(np.abs(V5[0] - T[0]))
    c = np.vdot(T[0], V5[0])
    return 1.0 - abs(c) ** 2 / (np.vdot(T[0], T[0]).real * np.vdot(V5[0], V5[0]).real)


@pytest.mark.parametrize("R", [None, 5.2e-3])
def test_o9_mae_loss_gradients_match_finite_differences(orc, R):
    """The paper's D2NN loss (mean absolute error between the processed field and the free-space result):
    every gradient of the chain with loss_kind="mae" equals a central finite difference of mean |V5 - T| written out
    here; with both masks zero and no turbulence the loss is 0 (the minimum; the loss is not differentiable there)."""
    N, dx, lam = 16, 1e-3, 1e-6
    dz = np.array([3.0, 5.0, 4.0])
    kw = dict(win_order=8, win_sigma_frac=0.45)
    u0 = synth.gaussian_beam(N, dx, 4e-3, 1).astype(np.complex128)
    scr = synth.random_screens(N, 1, 3, 5, rms=1.0).astype(np.float64)
    th = synth.phase_masks(0, N, 2).astype(np.float64)
    r = o9.oracle_chain(orc, N, dx, lam, dz, u0, scr, th[0], th[1], kw, aperture_radius=R, loss_kind="mae")
    assert abs(r["loss"][0] - _loss(orc, N, dx, lam, dz, u0, scr, th[0], th[1], kw, R, "mae")) < 1e-15
    rng = np.random.default_rng(1)
    h = 1e-6
    for what in ("th1", "th2", "phi0", "phi2"):
        for _ in range(4):
            iy, ix = rng.integers(2, N - 2, 2)
            t1p, t1m, t2p, t2m, sp, sm_ = th[0].copy(), th[0].copy(), th[1].copy(), th[1].copy(), scr.copy(), scr.copy()
            if what == "th1":
                t1p[iy, ix] += h; t1m[iy, ix] -= h; g = r["g_th1"][0, iy, ix]
            elif what == "th2":
                t2p[iy, ix] += h; t2m[iy, ix] -= h; g = r["g_th2"][0, iy, ix]
            else:
                s = int(what[-1])
                sp[0, s, iy, ix] += h; sm_[0, s, iy, ix] -= h; g = r["g_phi"][0, s, iy, ix]
            fd = (_loss(orc, N, dx, lam, dz, u0, sp, t1p, t2p, kw, R, "mae")
                  - _loss(orc, N, dx, lam, dz, u0, sm_, t1m, t2m, kw, R, "mae")) / (2 * h)
            assert abs(fd - g) < 1e-6 * max(1e-4, abs(g)) + 1e-10, (what, iy, ix, fd, g)
    z = np.zeros((N, N))
    r0 = o9.oracle_chain(orc, N, dx, lam, dz, u0, np.zeros_like(scr), z, z, kw, aperture_radius=R, loss_kind="mae")
    assert r0["loss"][0] < 1e-15


@pytest.mark.parametrize("R", [None, 5.2e-3])
def test_o9_gradients_match_finite_differences(orc, R):
    N, dx, lam = 16, 1e-3, 1e-6
    dz = np.array([3.0, 5.0, 4.0])
    kw = dict(win_order=8, win_sigma_frac=0.45)
    u0 = synth.gaussian_beam(N, dx, 4e-3, 1).astype(np.complex128)
    scr = synth.random_screens(N, 1, 3, 5, rms=1.0).astype(np.float64)
    th = synth.phase_masks(0, N, 2).astype(np.float64)
    r = o9.oracle_chain(orc, N, dx, lam, dz, u0, scr, th[0], th[1], kw, aperture_radius=R)
    assert 0.0 < r["loss"][0] < 1.0
    rng = np.random.default_rng(0)
    h = 1e-6
    for what in ("th1", "th2", "phi0", "phi2"):
        for _ in range(4):
            iy, ix = rng.integers(2, N - 2, 2)
            t1p, t1m, t2p, t2m, sp, sm_ = th[0].copy(), th[0].copy(), th[1].copy(), th[1].copy(), scr.copy(), scr.copy()
            if what == "th1":
                t1p[iy, ix] += h; t1m[iy, ix] -= h; g = r["g_th1"][0, iy, ix]
            elif what == "th2":
                t2p[iy, ix] += h; t2m[iy, ix] -= h; g = r["g_th2"][0, iy, ix]
            else:
                s = int(what[-1])
                sp[0, s, iy, ix] += h; sm_[0, s, iy, ix] -= h; g = r["g_phi"][0, s, iy, ix]
            fd = (_loss(orc, N, dx, lam, dz, u0, sp, t1p, t2p, kw, R) - _loss(orc, N, dx, lam, dz, u0, sm_, t1m, t2m, kw, R)) / (2 * h)
            assert abs(fd - g) < 1e-6 * max(1e-3, abs(g)) + 1e-9, (what, iy, ix, fd, g)
    if R is None:   # mask 1 and the last screen share a plane: their gradients are the same map
        np.testing.assert_allclose(r["g_th1"][0], r["g_phi"][0, 2], rtol=1e-9, atol=1e-14)
    else:           # ... inside the aperture; outside it the mask sees no light
        inside = np.abs(orc.aperture(N, dx, R, np.ones((1, N, N), dtype=np.complex128))[0]) > 0
        np.testing.assert_allclose(r["g_th1"][0][inside], r["g_phi"][0, 2][inside], rtol=1e-9, atol=1e-14)
        assert np.all(r["g_th1"][0][~inside] == 0)


def test_adam_step_pins(orc):
    """orc.adam_step (PAPER.md:115's optimiser): the first step moves every coordinate by lr against the sign of its
    gradient (bias correction makes m_hat = g, v_hat = g^2); a constant gradient keeps doing so; on a quadratic the
    iterates approach the minimum; the batch axis is averaged."""
    rng = np.random.default_rng(1)
    g = rng.standard_normal((3, 4, 4))
    th0 = rng.standard_normal((4, 4))
    m, v, th = orc.adam_step(g, 0.01, 1, np.zeros((4, 4)), np.zeros((4, 4)), th0)
    gm = g.mean(axis=0)
    np.testing.assert_allclose(th, th0 - 0.01 * np.sign(gm), atol=1e-7)
    np.testing.assert_allclose(m, 0.1 * gm)
    np.testing.assert_allclose(v, 0.001 * gm * gm)
    for t in range(2, 6):
        m, v, th2 = orc.adam_step(g, 0.01, t, m, v, th)
        np.testing.assert_allclose(th2, th - 0.01 * np.sign(gm), atol=1e-6)
        th = th2
    x, m, v = np.full((1, 1), 5.0), np.zeros((1, 1)), np.zeros((1, 1))
    for t in range(1, 2001):
        m, v, x = orc.adam_step(2 * (x - 1.0)[None], 0.05, t, m, v, x)
    assert abs(x[0, 0] - 1.0) < 1e-2
