"""P1, P1b, P5, P7, P8 -- pins for the oracle's split-step propagation (O6), adjoint (O7),
statistics (O8) and config-4 helpers (O9)."""
import numpy as np
import pytest

from paper_2604_07248_b200 import synth
from tests.util import paper_constants


def _gauss_q(N, dx, w0, lam, z):
    """Paraxial Gaussian beam (carrier exp(ikz) dropped): U = 1/(1+iz/zR) exp(-r^2/(w0^2 (1+iz/zR)))."""
    x = synth.coords(N, dx)
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    zR = np.pi * w0 * w0 / lam
    q = 1 + 1j * z / zR
    return np.exp(-r2 / (w0 * w0 * q)) / q


def test_vacuum_gaussian_width_and_field(orc):
    """P1: w2(z) = w0 sqrt(1 + (z/zR)^2) (north_star; PAPER.md:412 W(z) with theta0 = lambda/(pi w0), Q18),
    and the whole complex field against the paraxial closed form (fixes the sign of H)."""
    N, dx, lam, w0, L, S = 256, 1e-3, 1.55e-6, 2e-2, 1000.0, 5
    u0 = synth.gaussian_beam(N, dx, w0, 1)
    dz = np.full(S, L / S)
    u = orc.propagate(N, dx, lam, dz, u0)
    st = orc.beam_stats(N, dx, u)[0]
    zR = np.pi * w0 * w0 / lam
    w_th = w0 * np.sqrt(1 + (L / zR) ** 2)
    theta0 = lam / (np.pi * w0)
    assert abs(w_th - np.sqrt(w0 ** 2 + (theta0 * L) ** 2)) < 1e-15          # same closed form
    assert abs(st["w2"] / w_th - 1) < 1e-9
    assert abs(st["cx"]) < 1e-12 and abs(st["cy"]) < 1e-12
    ref = _gauss_q(N, dx, w0, lam, L)
    assert np.linalg.norm(u[0] - ref) / np.linalg.norm(ref) < 2e-7      # input is rounded to complex64
    # one step of L == S steps of L/S (H is a one-parameter group)
    u1 = orc.propagate(N, dx, lam, [L], u0)
    assert np.abs(u1 - u).max() < 1e-12
    # the stats of the input itself: power = pi w0^2 / 2, w2 = w0, I_axis = 1
    s0 = orc.beam_stats(N, dx, u0)[0]
    assert abs(s0["power"] / (np.pi * w0 * w0 / 2) - 1) < 1e-7              # complex64 input
    assert abs(s0["w2"] / w0 - 1) < 1e-7 and abs(s0["I_axis"] - 1) < 1e-6


def test_power_conservation_in_vacuum(orc):
    """P1b: Parseval -- |H| = 1, window off => sum |U|^2 is constant."""
    N, dx, lam = 64, 1e-3, 1e-6
    u0 = synth.random_field(N, 2, 3)
    for h_kind in (orc.H_FRESNEL, orc.H_ANGULAR_SPECTRUM):
        u = orc.propagate(N, dx, lam, [7.0, 13.0, 2.0], u0, h_kind=h_kind)
        p0 = np.sum(np.abs(u0.astype(np.complex128)) ** 2, axis=(1, 2))
        p1 = np.sum(np.abs(u) ** 2, axis=(1, 2))
        np.testing.assert_allclose(p1, p0, rtol=1e-13)
    # screens are pure phase: power still conserved
    scr = synth.random_screens(N, 2, 3, 1)
    u = orc.propagate(N, dx, lam, [7.0, 13.0, 2.0], u0, scr)
    np.testing.assert_allclose(np.sum(np.abs(u) ** 2, axis=(1, 2)), p0, rtol=1e-13)


def test_angular_spectrum_reduces_to_fresnel_when_paraxial(orc):
    """Eq.6 with the carrier removed (Q2) -> Fresnel H for kappa << k."""
    N, dx, lam, w0 = 128, 1e-3, 1.0e-6, 1e-2
    u0 = synth.gaussian_beam(N, dx, w0, 1)
    a = orc.propagate(N, dx, lam, [50.0, 50.0], u0, h_kind=orc.H_ANGULAR_SPECTRUM)
    f = orc.propagate(N, dx, lam, [50.0, 50.0], u0, h_kind=orc.H_FRESNEL)
    assert np.linalg.norm(a - f) / np.linalg.norm(f) < 1e-6
    # refractive index: lambda/n0 in the medium
    m = orc.propagate(N, dx, lam, [100.0], u0, n0=1.33)
    v = orc.propagate(N, dx, lam / 1.33, [100.0], u0)
    assert np.abs(m - v).max() < 1e-13


@pytest.mark.parametrize("mx,my,n0", [(5, 3, 1.0), (-7, 2, 1.0), (4, -4, 1.33)])
def test_angular_spectrum_non_paraxial_plane_wave(orc, mx, my, n0):
    """The non-paraxial term of Eq.6: a tilted plane wave exp(i 2 pi (mx ix + my iy)/N), periodic on the
    grid, with |kappa0| ~ 0.5 k is an eigenfunction of the step and must come out multiplied by
    exp(i dz (sqrt(k^2 - kappa0^2) - k)), k = 2 pi n0 / lambda (carrier removed, Q2).  The phase is evaluated here from
    Eq.6 itself with 50-digit arithmetic (mpmath); dz is chosen so that the Fresnel kernel is off by several radians,
    i.e. the test fails if the oracle falls back to the paraxial form or drops the square root."""
    import mpmath as mp
    mp.mp.dps = 50
    N, lam = 64, 1.0e-6
    dx = lam / n0 * 11.5 / N                                  # |f| = hypot(mx, my)/(N dx) ~ 0.5 n0/lambda for hypot ~ 5.8
    dz = 100.0 * lam
    iy, ix = np.mgrid[0:N, 0:N]
    u0 = np.exp(2j * np.pi * (mx * ix + my * iy) / N)[None]
    u = orc.propagate(N, dx, lam, [dz], u0, n0=n0, h_kind=orc.H_ANGULAR_SPECTRUM)
    k = 2 * mp.pi * mp.mpf(n0) / mp.mpf(lam)
    kap2 = (2 * mp.pi) ** 2 * (mp.mpf(mx) ** 2 + mp.mpf(my) ** 2) / (mp.mpf(N) * mp.mpf(dx)) ** 2
    assert 0.15 < float(kap2 / k ** 2) < 0.5                  # far from paraxial, still propagating
    ang = mp.mpf(dz) * (mp.sqrt(k ** 2 - kap2) - k)
    ang_fresnel = -mp.mpf(dz) * kap2 / (2 * k)
    assert abs(float(ang - ang_fresnel)) > 1.0                # > 1 rad away from the Fresnel phase
    factor = complex(mp.cos(ang), mp.sin(ang))
    assert np.abs(u[0] - factor * u0[0]).max() < 1e-10
    # two half steps compose (the phase is linear in dz), and the adjoint step undoes it (|H| = 1)
    u2 = orc.propagate(N, dx, lam, [dz / 2, dz / 2], u0, n0=n0, h_kind=orc.H_ANGULAR_SPECTRUM)
    assert np.abs(u2 - u).max() < 1e-10
    back = orc.propagate_adjoint(N, dx, lam, [dz], u, n0=n0, h_kind=orc.H_ANGULAR_SPECTRUM)
    assert np.abs(back - u0).max() < 1e-10


def test_tilt_screen_steers_the_beam(orc):
    """Sign of exp(+i phi) (Eq.1) and axis order: a prism phi = 2 pi ft x placed
    after step 1 moves the centroid by +lambda ft dz2 in x only."""
    N, dx, lam, w0 = 256, 1e-3, 1.0e-6, 1.5e-2
    u0 = synth.gaussian_beam(N, dx, w0, 1)
    x = synth.coords(N, dx)
    ft = 20.0                                                   # cycles/m
    phi = np.broadcast_to(2 * np.pi * ft * x[None, :], (N, N))
    scr = np.stack([phi, np.zeros((N, N))])[None]               # [B=1][S=2]
    u = orc.propagate(N, dx, lam, [100.0, 800.0], u0, scr)
    st = orc.beam_stats(N, dx, u)[0]
    assert abs(st["cx"] - lam * ft * 800.0) < 1e-9 and abs(st["cy"]) < 1e-12
    # shared stack (stride 0) gives the same result for every field
    u2 = orc.propagate(N, dx, lam, [100.0, 800.0], np.concatenate([u0, u0]), scr[0], shared_screens=True)
    assert np.abs(u2[0] - u[0]).max() == 0 and np.abs(u2[1] - u[0]).max() == 0
    # trailing vacuum step: S = n_steps - 1
    u3 = orc.propagate(N, dx, lam, [100.0, 800.0], u0, scr[:, :1])
    st3 = orc.beam_stats(N, dx, u3)[0]
    assert abs(st3["cx"] - lam * ft * 800.0) < 1e-9


def test_window_definition(orc):
    """Q12: W = exp(-((x^2+y^2)/sigma^2)^(p/2)), sigma = sigma_frac N dx, applied after every step."""
    N, dx, lam = 64, 1e-3, 1e-6
    u0 = synth.plane_wave(N, 1)
    u = orc.propagate(N, dx, lam, [1.0], u0, win_order=16, win_sigma_frac=0.47)
    x = synth.coords(N, dx)
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    W = np.exp(-(r2 / (0.47 * N * dx) ** 2) ** 8)
    np.testing.assert_allclose(u[0], W, atol=1e-13)              # plane wave is an eigenfunction of H (H(0)=1)
    u = orc.propagate(N, dx, lam, [1.0, 1.0], u0, win_order=4, win_sigma_frac=0.3)
    assert abs(abs(u[0, N // 2, N // 2]) - 1) < 1e-3 and abs(u[0, 0, 0]) < 1e-3


@pytest.mark.slow
def test_weak_plane_wave_scintillation_matches_rytov(orc):
    """P5: config-2 geometry at Cn2 = 1e-15 (weak): spatial SI of |U|^2 = discrete-screen Rytov sum
    2.25 k^(7/6) sum_j Cn2 dz_j d_j^(5/6), d_j = distance screen j -> receiver (Q11, Q13); its
    continuum limit is the paper's constant-Cn2 value 1.23 Cn2 k^(7/6) L^(11/6) (S19: 3.27 * 3/8)."""
    c = paper_constants()
    assert abs(c["rytov_const"] * 3 / 8 - c["si_weak_const"]) < 0.005      # S19 -> 1.23 for constant Cn2
    wl = synth.CONFIGS[2]
    N, dx, lam, S, L, cn2, nreal = wl.N, wl.dx, wl.lam, wl.S, wl.L, 1e-15, 8
    k = 2 * np.pi / lam
    hi, _ = synth.noise_batch(2, 0, nreal, S, N, 0)
    scr, _, _ = orc.make_screens(N, dx, orc.Psd(kind=orc.PSD_KOLMOGOROV), lam, [cn2] * S, wl.dz, 0, hi, None,
                                 keep_spectrum=False)
    u = orc.propagate(N, dx, lam, wl.dz, synth.plane_wave(N, nreal), scr)
    st = orc.beam_stats(N, dx, u, roi_frac=1.0)
    si = np.mean([s["roi_n"] * s["roi_sumI2"] / s["roi_sumI"] ** 2 - 1 for s in st])
    d = L - np.arange(1, S + 1) * L / S
    rytov_disc = 2.25 * k ** (7 / 6) * np.sum(cn2 * wl.dz * d ** (5 / 6))
    assert abs(si / rytov_disc - 1) < 0.05, (si, rytov_disc)
    cont = c["si_weak_const"] * cn2 * k ** (7 / 6) * L ** (11 / 6)
    assert abs(rytov_disc / cont - 1) < 0.12                    # 10 screens, last one in the receiver plane


@pytest.mark.parametrize("h_kind", [0, 1])
def test_adjoint_identity(orc, h_kind):
    """P7: <A x, y> = <x, A^H y> with random x, y, 3 random screens, window on."""
    N, dx, lam = 32, 1e-3, 1e-6
    dz = [5.0, 9.0, 4.0, 2.0]
    scr = synth.random_screens(N, 2, 3, 5)
    x = synth.random_field(N, 2, 1)
    y = synth.random_field(N, 2, 2)
    kw = dict(win_order=8, win_sigma_frac=0.4, h_kind=h_kind)
    Ax = orc.propagate(N, dx, lam, dz, x, scr, **kw)
    AHy = orc.propagate_adjoint(N, dx, lam, dz, y, scr, **kw)
    for b in range(2):
        lhs = np.vdot(y[b].astype(np.complex128), Ax[b])        # <y, A x>
        rhs = np.vdot(AHy[b], x[b].astype(np.complex128))       # <A^H y, x>
        assert abs(lhs - rhs) < 1e-12 * abs(lhs)


def test_phase_gradient_matches_finite_differences(orc):
    """P8: l = sum |U_out - T|^2; G_out = 2 (U_out - T); dl/dphi_j = Im(G_j conj(U_j))."""
    N, dx, lam = 16, 1e-3, 1e-6
    dz = [3.0, 6.0, 4.0]
    scr = synth.random_screens(N, 1, 3, 7).astype(np.float64)
    x = synth.random_field(N, 1, 3)
    T = synth.random_field(N, 1, 4).astype(np.complex128)
    kw = dict(win_order=8, win_sigma_frac=0.45)

    def loss(s):
        return np.sum(np.abs(orc.propagate(N, dx, lam, dz, x, s, **kw) - T) ** 2)
    out, planes = orc.propagate(N, dx, lam, dz, x, scr, return_planes=True, **kw)
    np.testing.assert_array_equal(planes[:, -1], out)
    g_in, grad = orc.propagate_adjoint(N, dx, lam, dz, 2 * (out - T), scr, planes=planes, **kw)
    rng = np.random.default_rng(0)
    for _ in range(8):
        j, iy, ix = rng.integers(0, 3), rng.integers(0, N), rng.integers(0, N)
        h = 1e-6
        sp, sm = scr.copy(), scr.copy()
        sp[0, j, iy, ix] += h
        sm[0, j, iy, ix] -= h
        fd = (loss(sp) - loss(sm)) / (2 * h)
        assert abs(fd - grad[0, j, iy, ix]) < 1e-6 * max(1.0, abs(fd)), (j, iy, ix, fd, grad[0, j, iy, ix])
    # gradient with respect to the input field: G_in = A^H G_out (real-pair convention)
    h = 1e-6
    for (iy, ix) in [(3, 4), (8, 8)]:
        for d, pick in ((1.0, np.real), (1j, np.imag)):
            xp, xm = x.astype(np.complex128).copy(), x.astype(np.complex128).copy()
            xp[0, iy, ix] += h * d
            xm[0, iy, ix] -= h * d
            fd = (np.sum(np.abs(orc.propagate(N, dx, lam, dz, xp, scr, **kw) - T) ** 2)
                  - np.sum(np.abs(orc.propagate(N, dx, lam, dz, xm, scr, **kw) - T) ** 2)) / (2 * h)
            assert abs(fd - pick(g_in[0, iy, ix])) < 1e-6 * max(1.0, abs(fd))


def test_beam_stats_closed_forms(orc):
    """O8 on fields with known moments."""
    N, dx = 128, 2e-3
    x = synth.coords(N, dx)
    X, Y = np.meshgrid(x, x)
    wx, wy, x0, y0 = 0.03, 0.02, 0.011, -0.007
    # elliptical, rotated-free Gaussian: sxx = wx^2/4, syy = wy^2/4
    u = np.exp(-((X - x0) ** 2) / wx ** 2 - ((Y - y0) ** 2) / wy ** 2)[None].astype(np.complex128)
    st = orc.beam_stats(N, dx, u, roi_frac=0.25)[0]
    assert abs(st["cx"] - x0) < 1e-9 and abs(st["cy"] - y0) < 1e-9
    assert abs(st["sxx"] / (wx ** 2 / 4) - 1) < 1e-8 and abs(st["syy"] / (wy ** 2 / 4) - 1) < 1e-8
    assert abs(st["sxy"]) < 1e-12
    assert abs(st["w2"] / np.sqrt((wx ** 2 + wy ** 2) / 2) - 1) < 1e-8
    assert abs(st["power"] / (np.pi * wx * wy / 2) - 1) < 1e-8
    assert st["roi_n"] == (N // 4) ** 2
    # correlated moments: rotate by 45 degrees -> sxy = (wx^2 - wy^2)/8
    Xr, Yr = (X + Y) / np.sqrt(2), (Y - X) / np.sqrt(2)
    u = np.exp(-(Xr ** 2) / wx ** 2 - (Yr ** 2) / wy ** 2)[None].astype(np.complex128)
    st = orc.beam_stats(N, dx, u)[0]
    assert abs(st["sxy"] / ((wx ** 2 - wy ** 2) / 8) - 1) < 1e-7
    # spatial scintillation index of I = 1 + m cos(2 pi 4 x / (N dx)) over the full grid: m^2/2 (S25)
    m = 0.3
    I = 1 + m * np.cos(2 * np.pi * 4 * X / (N * dx))
    st = orc.beam_stats(N, dx, np.sqrt(I)[None].astype(np.complex128) * np.exp(0.3j), roi_frac=1.0)[0]
    si = st["roi_n"] * st["roi_sumI2"] / st["roi_sumI"] ** 2 - 1
    assert abs(si - m * m / 2) < 1e-12 and st["roi_n"] == N * N
    # ROI bookkeeping: h = floor(roi_frac N / 2); h = 0 -> the on-axis pixel
    st = orc.beam_stats(N, dx, u, roi_frac=0.0)[0]
    assert st["roi_n"] == 1 and abs(st["roi_sumI"] - st["I_axis"]) < 1e-15


def test_welford_matches_two_pass(orc):
    """Welford's running variance of the intensity; SI = M2/(n-1)/mean^2 (unbiased)."""
    N, M = 16, 12
    u = synth.random_field(N, M, 9)
    mean = np.zeros((N, N))
    M2 = np.zeros((N, N))
    cnt = 0
    cnt = orc.welford(N, u[:5], mean, M2, cnt)
    cnt = orc.welford(N, u[5:], mean, M2, cnt)
    I = np.abs(u.astype(np.complex128)) ** 2
    assert cnt == M
    np.testing.assert_allclose(mean, I.mean(0), rtol=1e-12)
    np.testing.assert_allclose(M2 / (cnt - 1), I.var(0, ddof=1), rtol=1e-11)


def test_centered_dft_and_mask_helpers(orc):
    """O9: F_c = fftshift o fft2 o ifftshift / N (unitary); phase_mul; phase_grad."""
    N = 32
    u = synth.random_field(N, 2, 11).astype(np.complex128)
    ref = np.fft.fftshift(np.fft.fft2(np.fft.ifftshift(u, axes=(1, 2))), axes=(1, 2)) / N
    F = orc.dft2_centered(N, u)
    np.testing.assert_allclose(F, ref, atol=1e-12)
    np.testing.assert_allclose(orc.dft2_centered(N, F, inverse=True), u, atol=1e-12)
    assert abs(np.sum(np.abs(F) ** 2) / np.sum(np.abs(u) ** 2) - 1) < 1e-13
    # a centred Gaussian maps to a real positive centred Gaussian (no checkerboard sign)
    g = synth.gaussian_beam(N, 1.0, 4.0, 1).astype(np.complex128)
    G = orc.dft2_centered(N, g)
    assert np.abs(G.imag).max() < 1e-12 and G.real.min() > -1e-6 and np.argmax(G.real) == (N // 2) * N + N // 2
    th = synth.phase_masks(0, N, 1)[0].astype(np.float64)
    np.testing.assert_allclose(orc.phase_mul(N, th, u), u * np.exp(1j * th), atol=1e-13)
    np.testing.assert_allclose(orc.phase_mul(N, th, u, sign=-1.0), u * np.exp(-1j * th), atol=1e-13)
    v = synth.random_field(N, 2, 12).astype(np.complex128)
    np.testing.assert_allclose(orc.phase_grad(N, u, v), np.imag(u * np.conj(v)), atol=1e-13)


def test_circular_aperture(orc):
    """the receiver aperture.  Pixel count -> disc area, Gaussian energy fraction 1 - exp(-2 R^2/w^2),
    idempotent, nothing but 0 or the input."""
    N, dx, w0, R = 256, 1e-3, 3e-2, 4.05e-2
    u = synth.gaussian_beam(N, dx, w0, 2).astype(np.complex128) * (1 + 0.5j)
    out = orc.aperture(N, dx, R, u)
    inside = np.abs(out[0]) > 0
    assert abs(inside.sum() * dx * dx / (np.pi * R * R) - 1) < 2 * dx / R          # perimeter-cell bound
    frac = np.sum(np.abs(out[0]) ** 2) / np.sum(np.abs(u[0]) ** 2)
    assert abs(frac - (1 - np.exp(-2 * R * R / (w0 * w0)))) < 2e-3
    np.testing.assert_array_equal(orc.aperture(N, dx, R, out), out)
    np.testing.assert_array_equal(out[inside[None].repeat(2, 0)], u[inside[None].repeat(2, 0)])
    x = synth.coords(N, dx)
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    assert inside[r2 < (R - dx) ** 2].all() and not inside[r2 > (R + dx) ** 2].any()
