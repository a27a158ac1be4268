"""P2/P3 -- pins for the oracle's phase PSD (O2) and filter normalisation (O3).

What fixes them: the constants the paper prints (tests/golden/paper_constants.txt), the
structure-function law D(r) = 6.88 (r/r0)^(5/3) that north_star names (obtained here by
direct Hankel integration of the oracle's Phi^f, i.e. from the definition
D(r) = 2 int Phi^f(f) (1 - cos 2 pi f.r) d^2f), and the von Karman closed form."""
import numpy as np
import pytest
from scipy import integrate, special

from tests.util import paper_constants

LAM, CN2, DZ = 1.0e-6, 1.0e-14, 100.0


def _hankel_D(orc, psd, r):
    """D(r) = 4 pi int_0^inf Phi^f(f) (1 - J0(2 pi f r)) f df, integrated piecewise."""
    def g(f):
        return 4 * np.pi * orc.psd_f(psd, LAM, CN2, DZ, f)[0] * (1.0 - special.j0(2 * np.pi * f * r)) * f
    # head in the log variable (integrand ~ f^(1/3) for a pure power law: integrable at 0)
    total = integrate.quad(lambda u: g(np.exp(u)) * np.exp(u), np.log(1e-24 / r), np.log(1e-2 / r),
                           limit=400)[0]
    edges = np.concatenate([[1e-2 / r], np.arange(0.25, 60.25, 0.5) / r])
    for a, b in zip(edges[:-1], edges[1:]):
        total += integrate.quad(g, a, b, limit=200)[0]
    # tail beyond F = edges[-1]: J0 term averages out; int_F^inf Phi f df analytic for f^-11/3
    F = edges[-1]
    total += 4 * np.pi * orc.psd_f(psd, LAM, CN2, DZ, F)[0] * F ** (11 / 3) * (3 / 5) * F ** (-5 / 3)
    return total


def test_fried_parameter_is_S18(orc):
    c = paper_constants()
    k = 2 * np.pi / LAM
    expect = (c["fried_const"] * k * k * CN2 * DZ) ** c["fried_exponent"]
    assert abs(orc.r0(LAM, CN2, DZ) / expect - 1) < 1e-14


@pytest.mark.parametrize("r", [0.01, 0.05, 0.3])
def test_kolmogorov_psd_gives_688_law(orc, r):
    """0.023 r0^-5/3 f^-11/3 in cycles/m  <=>  D(r) = 6.88 (r/r0)^(5/3)  (Q4: units of S17)."""
    c = paper_constants()
    r0 = orc.r0(LAM, CN2, DZ)
    D = _hankel_D(orc, orc.Psd(kind=orc.PSD_KOLMOGOROV), r)
    law = c["structure_const"] * (r / r0) ** (5 / 3)
    # 0.023 is 0.0229 rounded (+0.45 %) and 6.88 is 6.884 rounded: agree to 1 %
    assert abs(D / law - 1) < 0.01, (D, law)


def test_psd_power_law_slope_and_constant(orc):
    c = paper_constants()
    psd = orc.Psd(kind=orc.PSD_KOLMOGOROV)
    f = np.array([0.5, 5.0, 50.0, 500.0])
    phi = orc.psd_f(psd, LAM, CN2, DZ, f)
    slope = np.diff(np.log(phi)) / np.diff(np.log(f))
    np.testing.assert_allclose(slope, -c["kolmogorov_alpha"], rtol=1e-12)
    r0 = orc.r0(LAM, CN2, DZ)
    assert abs(phi[0] / (c["psd_const"] * r0 ** (-5 / 3) * 0.5 ** (-11 / 3)) - 1) < 1e-13
    assert orc.psd_f(psd, LAM, CN2, DZ, 0.0)[0] == 0.0          # piston removed


def test_von_karman_closed_form_and_limits(orc):
    """S17 with f0 = 1/L0, fm = 1/l0 (kappa_m = 2 pi / l0); Kolmogorov limit."""
    c = paper_constants()
    L0, l0 = 10.0, 5e-3
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=L0, l0=l0)
    r0 = orc.r0(LAM, CN2, DZ)
    f = np.array([0.03, 0.1, 1.0, 30.0, 150.0])
    expect = c["psd_const"] * r0 ** (-5 / 3) * np.exp(-(f * l0) ** 2) / (f ** 2 + L0 ** -2) ** c["psd_exponent"]
    np.testing.assert_allclose(orc.psd_f(psd, LAM, CN2, DZ, f), expect, rtol=1e-13)
    # textbook kappa_m = 5.92/l0 through km_coeff
    psd2 = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=L0, l0=l0, km_coeff=5.92)
    fm = 5.92 / l0 / (2 * np.pi)
    expect2 = c["psd_const"] * r0 ** (-5 / 3) * np.exp(-(f / fm) ** 2) / (f ** 2 + L0 ** -2) ** (11 / 6)
    np.testing.assert_allclose(orc.psd_f(psd2, LAM, CN2, DZ, f), expect2, rtol=1e-13)
    # L0 -> inf, l0 -> 0 reduces to Kolmogorov (Table S1)
    big = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=1e9, l0=1e-9)
    np.testing.assert_allclose(orc.psd_f(big, LAM, CN2, DZ, f),
                               orc.psd_f(orc.Psd(kind=orc.PSD_KOLMOGOROV), LAM, CN2, DZ, f), rtol=1e-9)


def test_von_karman_structure_function_closed_form(orc):
    """Hankel integral of the oracle's von Karman PSD (l0 -> 0) vs the textbook closed form
    D(r) = 6.16 r0^-5/3 [0.6 k0^-5/3 - (r/(2 k0))^(5/6) K_5/6(k0 r)/Gamma(11/6)], k0 = 2 pi/L0."""
    L0 = 10.0
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=L0, l0=1e-7)
    r0 = orc.r0(LAM, CN2, DZ)
    k0 = 2 * np.pi / L0
    for r in (0.02, 0.2, 1.0):
        th = 6.16 * r0 ** (-5 / 3) * (0.6 * k0 ** (-5 / 3)
                                      - (r / (2 * k0)) ** (5 / 6) * special.kv(5 / 6, k0 * r) / special.gamma(11 / 6))
        D = _hankel_D(orc, psd, r)
        assert abs(D / th - 1) < 0.012, (r, D, th)


def test_ocean_spectrum_low_kappa_limit_and_projection(orc):
    """Nikishov (Q20, constants unpinned by the paper): as kappa*eta -> 0 the spectrum tends to
    0.388e-8 eps^-1/3 kappa^-11/3 chi_T (w^2 + 1 - 2w)/w^2, i.e. an alpha = 11/3 power law
    (Table S1 lower end); Phi^f = (2 pi)^3 k^2 dz Phi_n(2 pi f)."""
    chi_T, eps, w = 1e-7, 1e-5, -2.0
    psd = orc.Psd(kind=orc.PSD_OCEAN_NIKISHOV, chi_T=chi_T, eps=eps, w=w)
    lam, dz = 0.532e-6, 2.5
    k = 2 * np.pi / lam
    f = np.array([1e-5, 1e-4])
    kap = 2 * np.pi * f
    lim = 0.388e-8 * eps ** (-1 / 3) * kap ** (-11 / 3) * chi_T * (w * w + 1 - 2 * w) / (w * w)
    got = orc.psd_f(psd, lam, 0.0, dz, f)
    np.testing.assert_allclose(got, (2 * np.pi) ** 3 * k * k * dz * lim, rtol=5e-4)
    # log-slope stays inside Table S1's oceanic range [-15/3, -11/3] through the inertial range,
    # then the spectrum is cut off by dissipation
    ff = np.logspace(-2, 2.3, 40)
    ph = orc.psd_f(psd, lam, 0.0, dz, ff)
    assert np.all(ph > 0) and np.all(np.diff(ph) < 0)
    slope = np.diff(np.log(ph)) / np.diff(np.log(ff))
    assert abs(slope[0] + 11 / 3) < 0.02
    eta = (1e-18 / eps) ** 0.25
    assert abs(eta - 5.62e-4) < 1e-6                       # 0.562 mm for config 5
    # explicit eta is honoured
    psd_eta = orc.Psd(kind=orc.PSD_OCEAN_NIKISHOV, chi_T=chi_T, eps=eps, w=w, eta=eta)
    np.testing.assert_allclose(orc.psd_f(psd_eta, lam, 0.0, dz, ff), ph, rtol=1e-12)


def _nikishov_constants():
    import os
    from tests.util import GOLDEN
    out = {}
    with open(os.path.join(GOLDEN, "nikishov_constants.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if line:
                out[line[0]] = float(line[1])
    return out


@pytest.mark.parametrize("w", [-2.0, -0.5, -4.0])
def test_nikishov_against_retyped_constants(orc, w):
    """Q20: the oceanic spectrum is not in PAPER.md; its seven literature constants are re-typed in
    tests/golden/nikishov_constants.txt (with their source) and Phi_n is re-evaluated here from that file, term by
    term, at kappa eta = 0.01, 0.3, 3 and 10 (inertial range, the bump, the dissipation range, and the salinity-only
    tail where exp(-A_S delta) is all that is left), for three
    temperature / salinity balances w.  Every constant moves at least one of these values by far more than the
    tolerance: A_T / A_S / A_TS / D1 / D2 weigh in at kappa eta >= 0.3, C1 at 0.3, C0 everywhere."""
    c = _nikishov_constants()
    chi_T, eps = 1e-7, 1e-5
    lam, dz = 0.532e-6, 2.5
    k = 2 * np.pi / lam
    eta = (c["nu"] ** 3 / eps) ** 0.25
    psd = orc.Psd(kind=orc.PSD_OCEAN_NIKISHOV, chi_T=chi_T, eps=eps, w=w)
    for ke in (0.01, 0.3, 3.0, 10.0):
        kap = ke / eta
        delta = c["D1"] * ke ** (4.0 / 3.0) + c["D2"] * ke ** 2
        phin = (c["C0"] * eps ** (-1.0 / 3.0) * kap ** (-11.0 / 3.0) * (1.0 + c["C1"] * ke ** (2.0 / 3.0)) * chi_T / w ** 2
                * (w ** 2 * np.exp(-c["A_T"] * delta) + np.exp(-c["A_S"] * delta) - 2.0 * w * np.exp(-c["A_TS"] * delta)))
        want = (2 * np.pi) ** 3 * k * k * dz * phin                 # PAPER.md:346 (S14) projection, cycles/m
        got = orc.psd_f(psd, lam, 0.0, dz, kap / (2 * np.pi))[0]
        assert abs(got / want - 1) < 1e-12, (ke, got, want)
    # sensitivity of the sample points: a 1 % change of any constant moves some value by > 1e-4 relative
    def phi(cc, ke):
        delta = cc["D1"] * ke ** (4.0 / 3.0) + cc["D2"] * ke ** 2
        return (cc["C0"] * (1.0 + cc["C1"] * ke ** (2.0 / 3.0))
                * (w ** 2 * np.exp(-cc["A_T"] * delta) + np.exp(-cc["A_S"] * delta) - 2.0 * w * np.exp(-cc["A_TS"] * delta)))
    for name in ("C0", "C1", "A_T", "A_S", "A_TS", "D1", "D2"):
        cc = dict(c)
        cc[name] *= 1.01
        assert max(abs(phi(cc, ke) / phi(c, ke) - 1) for ke in (0.01, 0.3, 3.0, 10.0)) > 1e-4, name


def test_single_frequency_noise_returns_one_sinusoid(orc):
    """P3 (deterministic form): unit noise at one bin -> Re{ sqrt(Phi) df exp(+i 2 pi (kx ix + ky iy)/N) }
    (PAPER.md:359 S16: unnormalised inverse DFT, amplitude sqrt(Phi dfx dfy); Q3, Q6)."""
    N, dx = 32, 0.02
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    df = 1.0 / (N * dx)
    for (ky, kx, a, b) in [(0, 3, 1.0, 0.0), (5, 0, 0.0, 1.0), (N - 2, 7, 0.5, -2.0)]:
        noise = np.zeros((1, 1, N, N, 2), np.float32)
        noise[0, 0, ky, kx] = (a, b)
        scr, spec, _ = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], 0, noise, None)
        fy = (ky if ky < N // 2 else ky - N) * df
        fx = (kx if kx < N // 2 else kx - N) * df
        amp = np.sqrt(orc.psd_f(psd, LAM, CN2, DZ, np.hypot(fx, fy))[0]) * df
        iy, ix = np.mgrid[0:N, 0:N]
        expect = np.real((a + 1j * b) * amp * np.exp(2j * np.pi * (kx * ix + ky * iy) / N))
        np.testing.assert_allclose(scr[0, 0], expect, atol=1e-12 * amp * 10 + 1e-18)
        assert abs(spec[0, 0, ky, kx] - (a + 1j * b) * amp) < 1e-15 * amp * 10
    # DC noise is discarded
    noise = np.zeros((1, 1, N, N, 2), np.float32)
    noise[0, 0, 0, 0] = (3.0, 4.0)
    scr, _, _ = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], 0, noise, None)
    assert np.all(scr == 0.0)


# ---- general power-law media (PAPER.md:331 S12, Table S1) -------------------------------------------------
def _closed_form_D(K, alpha, r):
    """D(r) of Phi^f(f) = K f^-alpha (2 < alpha < 4): 4 pi K (2 pi r)^(alpha-2) int_0^inf x^(1-alpha) (1 - J0(x)) dx,
    with int_0^inf x^-p (1 - J0(x)) dx = pi / (2^p Gamma((p+1)/2)^2 sin(pi (p-1)/2)), p = alpha - 1."""
    p = alpha - 1.0
    integral = np.pi / (2.0 ** p * special.gamma((p + 1) / 2) ** 2 * np.sin(np.pi * (p - 1) / 2))
    return 4 * np.pi * K * (2 * np.pi * r) ** (alpha - 2) * integral


def test_closed_form_reproduces_688_law():
    """The closed form used below, fed the Kolmogorov constants, is the 6.88 law (an independent check of it)."""
    c = paper_constants()
    r0 = 0.1
    D = _closed_form_D(c["psd_const"] * r0 ** (-5 / 3), 11 / 3, 0.05)
    assert abs(D / (c["structure_const"] * (0.05 / r0) ** (5 / 3)) - 1) < 0.01


@pytest.mark.parametrize("alpha", [3.5, 11 / 3, 3.9])
def test_power_law_psd_structure_function(orc, alpha):
    """kind = POWER_LAW: Phi^f(f) = (2 pi)^3 k^2 dz A (2 pi f)^-alpha; its structure function by direct Hankel
    integration equals the closed form C r^(alpha-2) (Table S1: beta + 1 = alpha - 2)."""
    A = 3.3e-16
    psd = orc.Psd(kind=orc.PSD_POWER_LAW, alpha=alpha, A=A)
    k = 2 * np.pi / LAM
    K = (2 * np.pi) ** (3 - alpha) * k * k * DZ * A
    f = np.array([0.7, 13.0])
    np.testing.assert_allclose(orc.psd_f(psd, LAM, 0.0, DZ, f), K * f ** (-alpha), rtol=1e-13)
    r = 0.05

    def g(x):                                                  # x = 2 pi f r
        ff = x / (2 * np.pi * r)
        return 4 * np.pi * orc.psd_f(psd, LAM, 0.0, DZ, ff)[0] * (1.0 - special.j0(x)) * ff / (2 * np.pi * r)
    # head x < 1e-2 from the series 1 - J0(x) = x^2/4 - x^4/64 (the integrand ~ x^(3-alpha) converges slowly at 0)
    x0 = 1e-2
    total = 4 * np.pi * K * (2 * np.pi * r) ** (alpha - 2) * (x0 ** (4 - alpha) / (4 * (4 - alpha)) - x0 ** (6 - alpha) / (64 * (6 - alpha)))
    edges = np.concatenate([[x0], np.arange(0.5, 400.5, 1.0) * np.pi])
    for a, b in zip(edges[:-1], edges[1:]):
        total += integrate.quad(g, a, b, limit=200)[0]
    X = edges[-1]                                              # tail: the J0 term averages out
    total += 4 * np.pi * K * (2 * np.pi * r) ** (alpha - 2) * X ** (2 - alpha) / (alpha - 2)
    assert abs(total / _closed_form_D(K, alpha, r) - 1) < 5e-3


def test_power_law_reduces_to_the_atmospheric_kinds(orc):
    """alpha = 11/3, A = 0.033 Cn2 is Kolmogorov / von Karman up to the printed constants: 0.033 (2 pi)^(-2/3) against
    0.023 x 0.423 (0.4 % apart, Q24), with the same outer / inner scale roll-offs."""
    f = np.array([0.05, 0.5, 5.0, 50.0, 400.0])
    ratio = 0.033 * (2 * np.pi) ** (-2 / 3) / (0.023 * 0.423)
    assert abs(ratio - 1) < 5e-3
    pl = orc.Psd(kind=orc.PSD_POWER_LAW, alpha=11 / 3, A=0.033 * CN2)
    np.testing.assert_allclose(orc.psd_f(pl, LAM, 0.0, DZ, f) / orc.psd_f(orc.Psd(kind=orc.PSD_KOLMOGOROV), LAM, CN2, DZ, f),
                               ratio, rtol=1e-12)
    pl = orc.Psd(kind=orc.PSD_POWER_LAW, alpha=11 / 3, A=0.033 * CN2, L0=10.0, l0=5e-3)
    vk = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    np.testing.assert_allclose(orc.psd_f(pl, LAM, 0.0, DZ, f) / orc.psd_f(vk, LAM, CN2, DZ, f), ratio, rtol=1e-12)
