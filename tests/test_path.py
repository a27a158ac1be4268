"""Host-side path description (ssp_hv57_cn2 / ssp_hv57_path; PAPER.md:393 S21, :375 S18, :380 S19): pins of the
oracle's closed forms, then the library's quadrature against them.  No GPU needed: these are host functions."""
import numpy as np
import pytest
from scipy import integrate

LAM = 1.064e-6


def test_oracle_hv57_pins(orc):
    # S21 at the ground and the printed coefficients
    assert abs(orc.hv57_cn2(0.0, 1.7e-14) - (2.7e-16 + 1.7e-14)) < 1e-30
    h = 12000.0
    expect = 0.00594 * (21 / 27) ** 2 * (1e-5 * h) ** 10 * np.exp(-12.0) + 2.7e-16 * np.exp(-8.0) + 1.7e-14 * np.exp(-12.0)
    assert abs(orc.hv57_cn2(h, 1.7e-14) / expect - 1) < 1e-14
    # closed-form slab integral against adaptive quadrature of the profile
    for a, b in ((0.0, 1500.0), (3000.0, 20000.0)):
        num = integrate.quad(lambda x: float(orc.hv57_cn2(x, 1e-14)), a, b, epsabs=0, epsrel=1e-12)[0]
        assert abs(orc.hv57_slab_integral(a, b, 1e-14) / num - 1) < 1e-10
    # nearly constant profile (V = 0, A = 0, L << 1500 m): S19 -> 1.23 Cn2 k^(7/6) L^(11/6), S18 -> (0.423 k^2 Cn2 L)^(-3/5)
    L = 5.0
    cn2, dz, ry, r0 = orc.hv57_path(0.0, L, 4, LAM, 0.0, V=0.0)
    k = 2 * np.pi / LAM
    assert abs(ry / (3.27 * 3 / 8 * 2.7e-16 * k ** (7 / 6) * L ** (11 / 6)) - 1) < 2e-3
    assert abs(r0 / (0.423 * k * k * 2.7e-16 * L) ** (-3 / 5) - 1) < 2e-3
    assert np.allclose(dz, L / 4) and abs(cn2.mean() / 2.7e-16 - 1) < 2e-3


@pytest.mark.parametrize("h0,L,n,A,V,gs", [(0.0, 1500.0, 10, 1.7e-14, 21.0, 0.0), (0.0, 20000.0, 40, 10 ** -15.5, 21.0, 0.0),
                                            (500.0, 5000.0, 7, 1e-13, 57.0, 100.0)])
def test_library_path_matches_oracle(orc, h0, L, n, A, V, gs):
    from paper_2604_07248_b200 import api, build
    build.build()
    gso = gs if gs > 0 else 1000.0
    cn2, dz, ry, r0 = api.hv57_path(h0, L, n, LAM, A, V, gs)
    cn2_o, dz_o, ry_o, r0_o = orc.hv57_path(h0, L, n, LAM, A, V, gso)
    np.testing.assert_allclose(cn2, cn2_o, rtol=1e-9)
    np.testing.assert_allclose(dz, dz_o, rtol=1e-15)
    assert abs(ry / ry_o - 1) < 1e-6 and abs(r0 / r0_o - 1) < 1e-9
    for h in (0.0, 123.4, 9000.0):
        assert abs(api.hv57_cn2(h, A, V, gs) / float(orc.hv57_cn2(h, A, V, gso)) - 1) < 1e-13
    with pytest.raises(api.SspError):
        api.hv57_path(h0, -1.0, n, LAM, A)
