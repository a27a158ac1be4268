"""P2, P4, P6 -- pins for the oracle's screen synthesis (O3-O4) and AR evolution (O5)."""
import numpy as np
import pytest
from scipy import special

from paper_2604_07248_b200 import synth
from tests.util import paper_constants

LAM, CN2, DZ = 1.0e-6, 1.0e-14, 100.0


def _freqs(N, dx):
    k = np.arange(N)
    return np.where(k < N // 2, k, k - N) / (N * dx)


def _structure_fn(p, kmax):
    """Sample structure function along x and y separations of k pixels."""
    D = np.zeros(kmax)
    for k in range(1, kmax):
        D[k] = 0.5 * np.mean((p[..., :, k:] - p[..., :, :-k]) ** 2) + \
               0.5 * np.mean((p[..., k:, :] - p[..., :-k, :]) ** 2)
    return D


def test_ensemble_structure_function(orc):
    """P2: ensemble D(r) of von Karman screens with 3 subharmonic levels against
    (i) the exact discrete expectation  E D(r) = 2 sum_k s_k^2 (1 - cos 2 pi f_k.r)  over the FFT
        grid plus the subharmonic frequencies (pins S16's normalisation: unnormalised inverse
        DFT, real part of N(0,1)+iN(0,1) coefficients, s_k = sqrt(Phi) df, df_p = df/3^p), and
    (ii) the continuous von Karman closed form (pins units/constant end to end, 12 %)."""
    N, dx, L0, l0, n_sh = 128, 0.01, 10.0, 5e-3, 3
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=L0, l0=l0)
    S, nreal, kmax = 10, 40, N // 4
    acc = np.zeros(kmax)
    for b in range(nreal):
        hi, sh = synth.noise_batch(7, 0, 1, S, N, n_sh, b0=b)
        scr, _, _ = orc.make_screens(N, dx, psd, LAM, [CN2] * S, [DZ] * S, n_sh, hi, sh, keep_spectrum=False)
        assert np.abs(scr.mean(axis=(-2, -1))).max() < 1e-9 * np.abs(scr).max()   # piston removed
        acc += _structure_fn(scr[0], kmax)
    D = acc / nreal

    f = _freqs(N, dx)
    df = 1.0 / (N * dx)
    fx, fy = np.meshgrid(f, f)
    s2 = orc.psd_f(psd, LAM, CN2, DZ, np.hypot(fx, fy)) * df * df
    r = np.arange(kmax) * dx
    expect = np.zeros(kmax)
    for k in range(1, kmax):
        ex = 2 * np.sum(s2 * (1 - np.cos(2 * np.pi * fx * r[k])))
        for p in range(1, n_sh + 1):
            dfp = df / 3 ** p
            for m in (-1, 0, 1):
                for n in (-1, 0, 1):
                    if m == 0 and n == 0:
                        continue
                    sp2 = orc.psd_f(psd, LAM, CN2, DZ, np.hypot(m * dfp, n * dfp))[0] * dfp * dfp
                    # average of x- and y- separations
                    ex += sp2 * ((1 - np.cos(2 * np.pi * m * dfp * r[k])) + (1 - np.cos(2 * np.pi * n * dfp * r[k])))
        expect[k] = ex
    ks = np.array([1, 2, 4, 8, 16, 31])
    ratio = D[ks] / expect[ks]
    # statistical error only (400 screens); subharmonic mean removal changes D by O(1/N^2)
    assert np.all(np.abs(ratio - 1) < 0.08), ratio

    r0 = orc.r0(LAM, CN2, DZ)
    k0 = 2 * np.pi / L0
    rr = r[ks[1:]]
    th = 6.16 * r0 ** (-5 / 3) * (0.6 * k0 ** (-5 / 3)
                                  - (rr / (2 * k0)) ** (5 / 6) * special.kv(5 / 6, k0 * rr) / special.gamma(11 / 6))
    assert np.all(np.abs(D[ks[1:]] / th - 1) < 0.12), D[ks[1:]] / th

    # north_star's 6.88 law holds for r << outer scale / grid cut-off, within the allowance
    c = paper_constants()
    law = c["structure_const"] * (r[2] / r0) ** (5 / 3)
    assert abs(D[2] / law - 1) < 0.25


def test_subharmonic_levels_match_paper(orc):
    """s = 3, level p samples frequencies df/3^p; 3 levels = 27x finer."""
    c = paper_constants()
    assert c["sh_scale"] ** c["sh_levels"] == c["sh_resolution_gain"]
    N, dx = 32, 0.05
    psd = orc.Psd(kind=orc.PSD_KOLMOGOROV)
    df = 1.0 / (N * dx)
    x = synth.coords(N, dx)
    X, Y = np.meshgrid(x, x)
    for p in (1, 2, 3):
        for (a, b) in [(2, 1), (1, 0), (0, 2), (2, 2)]:          # [a]<->y multiplier a-1, [b]<->x multiplier b-1
            nsh = np.zeros((1, 1, 3, 3, 3, 2), np.float32)
            nsh[0, 0, p - 1, a, b] = (0.75, -1.25)
            hi = np.zeros((1, 1, N, N, 2), np.float32)
            scr, _, shc = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], 3, hi, nsh)
            dfp = df / c["sh_scale"] ** p
            fxp, fyp = (b - 1) * dfp, (a - 1) * dfp
            amp = np.sqrt(orc.psd_f(psd, LAM, CN2, DZ, np.hypot(fxp, fyp))[0]) * dfp
            lo = np.real((0.75 - 1.25j) * amp * np.exp(2j * np.pi * (fxp * X + fyp * Y)))
            expect = lo - lo.mean()
            np.testing.assert_allclose(scr[0, 0], expect, atol=1e-11 * amp)
            assert abs(shc[0, 0, p - 1, a, b] - (0.75 - 1.25j) * amp) < 1e-14 * amp
    # the centre (0,0) draw is unused
    nsh = np.zeros((1, 1, 3, 3, 3, 2), np.float32)
    nsh[0, 0, :, 1, 1] = (5.0, 5.0)
    scr, _, _ = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], 3, np.zeros((1, 1, N, N, 2), np.float32), nsh)
    assert np.all(scr == 0.0)


def test_subharmonic_mean_is_product_of_geometric_sums(orc):
    """P4: mean over the grid of exp(i 2 pi (fx x + fy y)) = Mx My with
    M = (1/N) sum_i exp(i 2 pi f x_i), a finite geometric sum; the oracle removes the brute-force mean."""
    N, dx, p = 64, 0.01, 2
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    nsh = np.zeros((1, 1, 3, 3, 3, 2), np.float32)
    nsh[0, 0, p - 1, 2, 0] = (1.0, 0.5)                      # fy = +dfp, fx = -dfp
    hi = np.zeros((1, 1, N, N, 2), np.float32)
    scr, _, shc = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], 3, hi, nsh)
    dfp = 1.0 / (N * dx) / 3 ** p
    x = synth.coords(N, dx)

    def M(f):                                                # closed form of the geometric sum
        q = np.exp(2j * np.pi * f * dx)
        return np.exp(2j * np.pi * f * x[0]) * (1 - q ** N) / (1 - q) / N
    c = shc[0, 0, p - 1, 2, 0]
    mean_analytic = np.real(c * M(-dfp) * M(+dfp))
    X, Y = np.meshgrid(x, x)
    lo = np.real(c * np.exp(2j * np.pi * (-dfp * X + dfp * Y)))
    assert abs(lo.mean() - mean_analytic) < 1e-13 * abs(c)
    np.testing.assert_allclose(scr[0, 0], lo - mean_analytic, atol=1e-12 * abs(c))


def _mk(orc, N, dx, psd, n_sh, B, S, frame, cid=11):
    hi, sh = synth.noise_batch(cid, 0, B, S, N, n_sh, frame=frame)
    return hi, sh


def test_ar_recursion_identities(orc):
    """P6: a = 1 keeps the screen, a = 0 replaces it by the fresh one, and for v = 0 the real-space
    identity phi_{t+1} = a phi_t + sqrt(1-a^2) phi_fresh (north_star; Eq.5; Q8) holds."""
    N, dx, n_sh, B, S = 32, 0.02, 3, 2, 2
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    cn2, dz = [CN2, 2 * CN2], [DZ, 50.0]
    hi0, sh0 = _mk(orc, N, dx, psd, n_sh, B, S, 0)
    hi1, sh1 = _mk(orc, N, dx, psd, n_sh, B, S, 1)
    scr0, spec0, shc0 = orc.make_screens(N, dx, psd, LAM, cn2, dz, n_sh, hi0, sh0)
    fresh, _, _ = orc.make_screens(N, dx, psd, LAM, cn2, dz, n_sh, hi1, sh1)
    scale = np.abs(scr0).max()

    sp, sc = spec0.copy(), shc0.copy()
    out = orc.evolve_screens(N, dx, psd, LAM, cn2, dz, n_sh, 1.0, 0, 0, 0.0, hi1, sh1, sp, sc)
    np.testing.assert_allclose(out, scr0, atol=1e-12 * scale)
    sp, sc = spec0.copy(), shc0.copy()
    out = orc.evolve_screens(N, dx, psd, LAM, cn2, dz, n_sh, 0.0, 0, 0, 0.0, hi1, sh1, sp, sc)
    np.testing.assert_allclose(out, fresh, atol=1e-12 * scale)
    a = 0.99
    sp, sc = spec0.copy(), shc0.copy()
    out = orc.evolve_screens(N, dx, psd, LAM, cn2, dz, n_sh, a, 0, 0, 0.0, hi1, sh1, sp, sc)
    np.testing.assert_allclose(out, a * scr0 + np.sqrt(1 - a * a) * fresh, atol=1e-12 * scale)
    # the stored spectrum is what was synthesised
    np.testing.assert_allclose(orc.synthesize(N, dx, n_sh, sp, sc), out, atol=1e-12 * scale)
    with pytest.raises(RuntimeError):
        orc.evolve_screens(N, dx, psd, LAM, cn2, dz, n_sh, 1.5, 0, 0, 0.0, hi1, sh1, sp, sc)


def test_ar_wind_shift_is_circular_roll(orc):
    """Eq.4 (with its i; Q9): tau = exp(-i 2 pi T (fx vx + fy vy)) moves the
    high-frequency screen by +v T; an integer number of pixels is an exact circular roll."""
    N, dx, B, S = 32, 0.02, 1, 1
    psd = orc.Psd(kind=orc.PSD_KOLMOGOROV)
    hi0, _ = _mk(orc, N, dx, psd, 0, B, S, 0)
    hi1, _ = _mk(orc, N, dx, psd, 0, B, S, 1)
    scr0, spec0, _ = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], 0, hi0, None)
    sp = spec0.copy()
    T, vx, vy = 0.5, 3 * dx / 0.5, -2 * dx / 0.5             # +3 px in x, -2 px in y
    out = orc.evolve_screens(N, dx, psd, LAM, [CN2], [DZ], 0, 1.0, vx, vy, T, hi1, None, sp, None)
    expect = np.roll(np.roll(scr0[0, 0], 3, axis=1), -2, axis=0)
    np.testing.assert_allclose(out[0, 0], expect, atol=1e-11 * np.abs(scr0).max())


@pytest.mark.parametrize("p,a,b", [(1, 0, 2), (2, 2, 1), (3, 1, 0), (2, 0, 0)])
def test_ar_wind_on_subharmonics_is_the_closed_form(orc, p, a, b):
    """Q8 under wind (Eq.4 applied to the subharmonic coefficients of Eq.2): one subharmonic coefficient
    c at (fx, fy) = ((b-1) df_p, (a-1) df_p), zero grid noise, AR factor 1, wind (vx, vy) over T.  The evolved screen
    must be  Re{ c exp(-i 2 pi T (fx vx + fy vy)) exp(i 2 pi (fx x + fy y)) }  minus its mean -- the sinusoid moved by
    +v T -- with vx != vy and (a, b) off the diagonal, so an x/y swap, a dropped level scaling of df_p or a sign error
    in tau fails.  The expectation is written out here from the formula, not taken from the oracle."""
    N, dx, n_sh = 32, 0.05, 3
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    nsh = np.zeros((1, 1, n_sh, 3, 3, 2), np.float32)
    nsh[0, 0, p - 1, a, b] = (0.75, -1.25)
    zero = np.zeros((1, 1, N, N, 2), np.float32)
    _, spec, shc = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], n_sh, zero, nsh)
    c = shc[0, 0, p - 1, a, b]
    assert abs(c) > 0
    T, vx, vy = 0.37, 1.9, -0.8                              # v T = (0.70, -0.30) m: a fraction of the 43 m .. 14 m periods
    fresh_sh = np.zeros_like(nsh)
    fresh_sh[0, 0, :, :, :] = (3.0, -2.0)                    # a = 1: fresh draws must not enter
    out = orc.evolve_screens(N, dx, psd, LAM, [CN2], [DZ], n_sh, 1.0, vx, vy, T, zero, fresh_sh, spec, shc)
    dfp = 1.0 / (N * dx) / 3.0 ** p
    fx, fy = (b - 1) * dfp, (a - 1) * dfp
    x = synth.coords(N, dx)
    X, Y = np.meshgrid(x, x)
    tau = np.exp(-2j * np.pi * T * (fx * vx + fy * vy))
    lo = np.real(c * tau * np.exp(2j * np.pi * (fx * X + fy * Y)))
    np.testing.assert_allclose(out[0, 0], lo - lo.mean(), rtol=0, atol=1e-12 * abs(c))
    # the same statement as a shift: phi_new(x, y) = phi_old(x - vx T, y - vy T) before mean removal
    shifted = np.real(c * np.exp(2j * np.pi * (fx * (X - vx * T) + fy * (Y - vy * T))))
    np.testing.assert_allclose(lo, shifted, rtol=0, atol=1e-12 * abs(c))
    assert abs(shc[0, 0, p - 1, a, b] - c * tau) < 1e-14 * abs(c)           # the stored coefficient carries the tilt
    assert abs(tau - 1) > 0.01                                # the wind does something at this level


def test_ar_decorrelation_follows_a_power_n(orc):
    """P6 statistical: with v = 0, corr(phi_t, phi_{t+n}) -> a^n and the variance stays stationary
    (Pearson score, threshold 0.4; a = 0.99 crosses 0.4 at n ~ 91)."""
    c = paper_constants()
    a = 0.99
    assert abs(np.log(c["pearson_threshold"]) / np.log(a) - 91.2) < 0.1
    N, dx, B, S = 32, 0.02, 24, 1
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=1.0, l0=5e-3)   # small L0: many independent modes per screen
    a = 0.9
    hi0, sh0 = synth.noise_batch(12, 0, B, S, N, 0, frame=0)
    scr0, spec, _ = orc.make_screens(N, dx, psd, LAM, [CN2], [DZ], 0, hi0, None)
    var0 = scr0.var()
    for n in range(1, 11):
        hin, _ = synth.noise_batch(12, 0, B, S, N, 0, frame=n)
        scr = orc.evolve_screens(N, dx, psd, LAM, [CN2], [DZ], 0, a, 0, 0, 0.0, hin, None, spec, None)
        if n in (1, 5, 10):
            corr = np.mean([np.corrcoef(scr0[b, 0].ravel(), scr[b, 0].ravel())[0, 1] for b in range(B)])
            assert abs(corr - a ** n) < 0.06, (n, corr, a ** n)
    assert abs(scr.var() / var0 - 1) < 0.15


def test_imaginary_part_is_a_second_screen(orc):
    """orc.synthesize(part="im") (the part of the synthesis that Q3 discards).  Exact link to the pinned
    real-part path: Im(z) = Re(-i z), so the imaginary-part screens of noise n are the real-part screens of noise
    -i n = (b, -a), subharmonics and mean removal included.  Ensemble: same variance as the real part, and
    uncorrelated with it (a circular complex Gaussian spectrum)."""
    N, dx, n_sh, B, S = 32, 2e-3, 3, 200, 1
    psd = orc.Psd(kind=orc.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    rng = np.random.default_rng(11)
    hi = rng.standard_normal((B, S, N, N, 2), dtype=np.float32)
    sh = rng.standard_normal((B, S, n_sh, 3, 3, 2), dtype=np.float32)
    re, spec, shc = orc.make_screens(N, dx, psd, 1e-6, [1e-14], [100.0], n_sh, hi, sh)
    im = orc.synthesize(N, dx, n_sh, spec, shc, part="im")
    rot = lambda a: np.stack([a[..., 1], -a[..., 0]], axis=-1).astype(np.float32)      # n -> -i n
    re_rot, _, _ = orc.make_screens(N, dx, psd, 1e-6, [1e-14], [100.0], n_sh, rot(hi), rot(sh))
    np.testing.assert_allclose(im, re_rot, rtol=0, atol=1e-12 * np.abs(re).max())
    np.testing.assert_allclose(orc.synthesize(N, dx, n_sh, spec, shc), re, rtol=0, atol=1e-12 * np.abs(re).max())
    assert abs(im.var() / re.var() - 1) < 0.25
    corr = np.mean(re * im) / np.sqrt(re.var() * im.var())
    assert abs(corr) < 0.2, corr           # a few low-frequency modes dominate: ~1/sqrt(200 x few) sampling noise
    assert np.abs(im.mean(axis=(-2, -1))).max() < 1e-10 * np.abs(im).max() + 1e-9    # piston removed here too
