"""Screen placement (Sec. 2.4; Q17, Q28): pins of the oracle's routine to what the text and the
mathematics fix, then the library's routine (closed-form piece integrals) against the oracle's (adaptive quadrature).
Host functions only: no GPU needed."""
import numpy as np
import pytest

LAM = 1.55e-6
K = 2 * np.pi / LAM


def test_oracle_dz_max_is_the_nyquist_step(orc):
    """At dz = dz_max the phase of H_as (Eq. 6) advances by pi between the two outermost frequency
    samples of an axis (to O(1/N)), and by less everywhere else; paraxial limit N dx^2 n0 / lambda."""
    for N, dx, n0 in ((512, 5e-3, 1.0), (1024, 2e-5, 1.34), (256, 3e-6, 1.0)):
        dz = orc.dz_max_angular_spectrum(N, dx, LAM, n0)
        kap = 2 * np.pi * np.fft.fftshift(np.fft.fftfreq(N, dx))           # -pi/dx .. pi/dx - dkappa
        psi = dz * np.sqrt((n0 * K) ** 2 - kap ** 2)
        jump = np.abs(np.diff(psi))
        assert abs(jump.max() / np.pi - 1) < 3.0 / N and jump.argmax() == 0
        par = N * dx * dx * n0 / LAM
        assert dz <= par and abs(dz / par - 1) < (LAM / (2 * n0 * dx)) ** 2
    assert orc.dz_max_angular_spectrum(64, 0.5e-6, LAM) == 0.0                  # pi/dx beyond n0 k0: evanescent


def test_oracle_interval_rytov_pins(orc):
    # constant Cn2: S19 -> the plane-wave Rytov variance 1.23 Cn2 k^(7/6) d^(11/6) (3.27 * 3/8 = 1.226)
    d, cn = 1234.0, 3e-15
    v = orc.interval_rytov(lambda z: cn, 100.0, 100.0 + d, LAM)
    assert abs(v / (1.23 * cn * K ** (7 / 6) * d ** (11 / 6)) - 1) < 4e-3
    assert abs(v / (3.27 * 3 / 8 * cn * K ** (7 / 6) * d ** (11 / 6)) - 1) < 1e-11
    # a thin layer at distance s from the END of the interval contributes 3.27 k^(7/6) d^(5/6) (s/d)^(5/3) Cn2 dz:
    # a layer at the start of the interval counts fully, one at its end not at all (the weight of S19)
    eps = 1e-3
    for pos, wt in ((0.0, 1.0), (d / 2, 0.5 ** (5 / 3)), (d - eps, 0.0)):
        lay = lambda z: cn if pos <= z - 100.0 <= pos + eps else 0.0
        v = orc.interval_rytov(lay, 100.0, 100.0 + d, LAM, kinks=(100.0 + pos, 100.0 + pos + eps))
        assert abs(v - 3.27 * K ** (7 / 6) * d ** (5 / 6) * wt * cn * eps) < 1e-5 * 3.27 * K ** (7 / 6) * d ** (5 / 6) * cn * eps
    # the same S19 as the path integral of hv57_path (a different code path of the oracle)
    z = np.linspace(0.0, 3000.0, 3001)
    c = orc.hv57_cn2(z, 1.7e-14)
    ry = orc.hv57_path(0.0, 3000.0, 3, LAM, 1.7e-14)[2]
    assert abs(orc.interval_rytov(lambda x: np.interp(x, z, c), 0.0, 3000.0, LAM, z) / ry - 1) < 1e-6


def test_oracle_placement_constant_profile_closed_forms(orc):
    """Constant Cn2: variance of an interval = c d^(11/6), so every stage has a closed form."""
    L, cn, lim = 20000.0, 1e-15, 0.2
    c = 3.27 * 3 / 8 * cn * K ** (7 / 6)
    dmax = (lim / c) ** (6 / 11)                                                # 3525.75 m
    dz, cn2, ry, st = orc.place_screens([0, L], [cn, cn], [0, L], LAM, lim, 0.0, return_stages=True)
    m = int(np.ceil(np.log2(L / dmax)))
    # 1: halved m times; 2: no two neighbours fit (2 L / 2^m > dmax by minimality of m)
    assert np.allclose(st["split"], np.linspace(0, L, 2 ** m + 1)) and np.allclose(st["merged"], st["split"])
    # 3: first end = chord through (d1, c d1^(11/6)) and (2 d1, c (2 d1)^(11/6)) at the limit, d1 = L / 2^m
    d1 = L / 2 ** m
    v1, v2 = c * d1 ** (11 / 6), c * (2 * d1) ** (11 / 6)
    assert abs(st["fitted"][1] - (d1 + (lim - v1) / (v2 - v1) * d1)) < 1e-6
    # the variance is convex in d, so the chord is conservative: within the limit, and closer to it than stage 2 was
    assert np.all(ry <= lim * (1 + 1e-12)) and ry[:-1].min() > v1 * 1.5 and len(dz) < 2 ** m
    assert abs(dz.sum() - L) < 1e-9 and np.allclose(cn2, cn, rtol=1e-12)
    assert np.allclose(ry, c * dz ** (11 / 6), rtol=1e-10)
    assert len(dz) >= int(np.ceil(L / dmax))                                    # no placement can use fewer
    # 2: 64 fine intervals merge greedily into runs of floor(dmax / (L/64)) = 11
    dzf, _, _, stf = orc.place_screens([0, L], [cn, cn], np.linspace(0, L, 65), LAM, lim, 0.0, return_stages=True)
    run = int(dmax // (L / 64))
    assert np.allclose(np.diff(stf["merged"])[:-1], run * L / 64) and abs(dzf.sum() - L) < 1e-9
    # 4: an aliasing limit below the fitted lengths halves them
    dza, _, rya = orc.place_screens([0, L], [cn, cn], [0, L], LAM, lim, 1000.0)
    assert dza.max() <= 1000.0 and len(dza) == 4 * (len(dz) - 1) + int(2 ** np.ceil(np.log2(dz[-1] / 1000.0)))
    assert abs(dza.sum() - L) < 1e-9


def test_oracle_placement_hv57_invariants(orc):
    """Vertical HV5/7 path: every interval within both limits, the slabs tile the path, the slab means carry the
    profile's integral (closed form of the sampled profile's trapezoid), strong ground layer -> short first slabs."""
    z = np.linspace(0.0, 20000.0, 201)
    c = orc.hv57_cn2(z, 1.7e-14, 21.0, 100.0)
    dzm = orc.dz_max_angular_spectrum(512, 5e-3, LAM)
    for lim in (0.05, 0.01):
        dz, cn2, ry, st = orc.place_screens(z, c, [0.0, 20000.0], LAM, lim, dzm, return_stages=True)
        assert np.all(ry <= lim * (1 + 1e-9)) and np.all(dz <= dzm * (1 + 1e-12)) and abs(dz.sum() - 20000.0) < 1e-6
        trap = np.sum(0.5 * (c[1:] + c[:-1]) * np.diff(z))
        assert abs(np.sum(cn2 * dz) / trap - 1) < 1e-10
        assert dz[0] < dz[-1]
        mg = st["merged"]                                                       # stage 2 left no mergeable pair
        f = lambda x: np.interp(x, z, c)
        assert all(orc.interval_rytov(f, mg[i], mg[i + 2], LAM, z) > lim for i in range(len(mg) - 2))
    assert len(orc.place_screens(z, c, [0.0, 20000.0], LAM, 0.01, dzm)[0]) > len(
        orc.place_screens(z, c, [0.0, 20000.0], LAM, 0.05, dzm)[0])


CASES = [
    ([0.0, 20000.0], [1e-15, 1e-15], [0.0, 20000.0], 0.2, 0.0),
    ([0.0, 20000.0], [1e-15, 1e-15], list(np.linspace(0.0, 20000.0, 65)), 0.2, 1000.0),
    ("hv", None, [0.0, 20000.0], 0.05, 8258.0),
    ("hv", None, [0.0, 500.0, 2000.0, 6000.0, 20000.0], 0.013, 3000.0),
    ([0.0, 1000.0, 1100.0, 1200.0, 5000.0], [1e-16, 1e-16, 4e-14, 1e-16, 1e-16], [0.0, 5000.0], 0.03, 0.0),   # strong layer
]


@pytest.mark.parametrize("zp,cp,edges,lim,dzm", CASES)
def test_library_placement_matches_oracle(orc, zp, cp, edges, lim, dzm):
    from paper_2604_07248_b200 import api, build
    build.build()
    if isinstance(zp, str):
        zp = np.linspace(0.0, 20000.0, 201)
        cp = orc.hv57_cn2(zp, 1.7e-14, 21.0, 100.0)
    dz_o, cn2_o, ry_o = orc.place_screens(zp, cp, edges, LAM, lim, dzm)
    dz, cn2, ry = api.place_screens(zp, cp, edges, LAM, lim, dzm)
    assert len(dz) == len(dz_o)
    np.testing.assert_allclose(dz, dz_o, rtol=1e-8)
    np.testing.assert_allclose(cn2, cn2_o, rtol=1e-8)
    np.testing.assert_allclose(ry, ry_o, rtol=1e-8)


def test_library_dz_max_and_errors(orc):
    from paper_2604_07248_b200 import api, build
    build.build()
    for N, dx, n0 in ((512, 5e-3, 1.0), (1024, 2e-5, 1.34), (64, 0.5e-6, 1.0)):
        a, b = api.dz_max(N, dx, LAM, n0), orc.dz_max_angular_spectrum(N, dx, LAM, n0)
        assert a == b == 0.0 or abs(a / b - 1) < 1e-14
    with pytest.raises(api.SspError) as e:
        api.place_screens([0.0, 1.0], [1e-15, 1e-15], [0.0, 1.0, 0.5], LAM, 0.1)       # edges not ascending
    assert e.value.code == api.EINVAL
    with pytest.raises(api.SspError) as e:
        api.place_screens([0.0, 2e4], [1e-15, 1e-15], [0.0, 2e4], LAM, 0.2, 0.0, max_out=3)   # needs 6
    assert e.value.code == api.EWORKSPACE
    with pytest.raises(api.SspError):
        api.place_screens([0.0, 2e4], [1e-15, -1e-15], [0.0, 2e4], LAM, 0.2)          # negative Cn2
