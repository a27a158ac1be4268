"""P0 -- pins for the oracle's DFT routines (oracle/orc.c) against things other than itself:
the DFT matrix written out, numpy's pocketfft, impulse / single-tone closed forms, Parseval."""
import numpy as np
import pytest


def _dft_matrix(n, sign):
    k = np.arange(n)
    return np.exp(sign * 2j * np.pi * np.outer(k, k) / n)


@pytest.mark.parametrize("n", [2, 4, 8, 16, 32])
@pytest.mark.parametrize("sign", [-1, +1])
def test_naive_dft_is_the_dft_matrix(orc, n, sign):
    rng = np.random.default_rng(n)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    np.testing.assert_allclose(orc.dft1d_naive(a, sign), _dft_matrix(n, sign) @ a, rtol=0, atol=1e-12)


@pytest.mark.parametrize("n", [64, 128, 512, 1024, 4096])
@pytest.mark.parametrize("sign", [-1, +1])
def test_radix2_matches_numpy(orc, n, sign):
    rng = np.random.default_rng(n + 1)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    ref = np.fft.fft(a) if sign < 0 else np.fft.ifft(a) * n
    got = orc.fft1d(a, sign)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) < 1e-14


@pytest.mark.parametrize("n", [64, 256])
def test_radix2_matches_naive_definition(orc, n):
    rng = np.random.default_rng(5)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert np.abs(orc.fft1d(a, -1) - orc.dft1d_naive(a, -1)).max() < 1e-11


@pytest.mark.parametrize("n", [16, 64, 1024])
def test_impulse_tone_parseval(orc, n):
    e = np.zeros(n, complex)
    e[3] = 1.0
    # impulse at n0=3 -> exp(-i 2 pi k 3 / n)
    np.testing.assert_allclose(orc.fft1d(e, -1), np.exp(-2j * np.pi * np.arange(n) * 3 / n), atol=1e-12)
    # single tone exp(+i 2 pi 5 j / n) -> n * delta[k-5] (forward sign is minus)
    tone = np.exp(2j * np.pi * 5 * np.arange(n) / n)
    out = orc.fft1d(tone, -1)
    expect = np.zeros(n, complex)
    expect[5] = n
    np.testing.assert_allclose(out, expect, atol=1e-9)
    rng = np.random.default_rng(0)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert abs(np.sum(np.abs(orc.fft1d(a)) ** 2) - n * np.sum(np.abs(a) ** 2)) < 1e-9 * n * n


@pytest.mark.parametrize("n", [8, 32, 64, 256])
def test_fft2d_matches_numpy_and_axes(orc, n):
    rng = np.random.default_rng(n)
    a = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    ref = np.fft.fft2(a)
    assert np.linalg.norm(orc.fft2d(a, -1) - ref) / np.linalg.norm(ref) < 1e-13
    ref = np.fft.ifft2(a) * n * n
    assert np.linalg.norm(orc.fft2d(a, +1) - ref) / np.linalg.norm(ref) < 1e-13
    # a tone along x only (ix varies fastest) lands in column kx, row ky=0: catches a transpose
    ix = np.arange(n)
    t = np.broadcast_to(np.exp(2j * np.pi * 3 * ix / n), (n, n)).copy()
    out = orc.fft2d(t, -1)
    assert abs(out[0, 3] - n * n) < 1e-8 and abs(out[3, 0]) < 1e-8


def test_fft_roundtrip(orc):
    rng = np.random.default_rng(1)
    a = rng.standard_normal((128, 128)) + 1j * rng.standard_normal((128, 128))
    b = orc.fft2d(orc.fft2d(a, -1), +1) / 128 ** 2
    assert np.abs(a - b).max() < 1e-12
