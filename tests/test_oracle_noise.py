"""Pins of the oracle's counter-based Gaussian noise (oracle/orc.py: philox4x32_10, noise; Q29).  The paper fixes
only the law of the draws ("unit-variance complex Gaussian", PAPER.md:359 S16; Q3: Re and Im each N(0, 1), independent), so
the pins are that law, independence across draws / streams / seeds, and the generator's structure (bijective rounds, full
64-bit draw index, avalanche)."""
import os

import numpy as np
from scipy import stats

from tests.util import GOLDEN

NS = 1 << 20


def test_noise_law(orc):
    z = orc.noise(2604, 7248, NS)
    for x in (z.real, z.imag):
        assert abs(x.mean()) < 4 / np.sqrt(NS) and abs(x.var() - 1) < 4 * np.sqrt(2.0 / NS)
        assert abs(stats.skew(x)) < 4 * np.sqrt(6.0 / NS) and abs(stats.kurtosis(x)) < 4 * np.sqrt(24.0 / NS)
        assert stats.kstest(x, "norm").pvalue > 1e-3
    assert abs(np.mean(z.real * z.imag)) < 4 / np.sqrt(NS)                      # Re, Im uncorrelated
    assert abs(np.mean(np.abs(z) ** 2) - 2) < 4 * 2 / np.sqrt(NS)                # E|z|^2 = 2 (Q3)
    assert stats.kstest(np.abs(z) ** 2, "expon", args=(0, 2)).pvalue > 1e-3      # |z|^2 ~ Exp(mean 2)
    assert stats.kstest(np.angle(z), "uniform", args=(-np.pi, 2 * np.pi)).pvalue > 1e-3
    # 23-bit uniforms: the radius is finite and at most sqrt(-2 ln 2^-24)
    assert np.all(np.isfinite(z.view(np.float64))) and np.abs(z).max() <= np.sqrt(48 * np.log(2)) + 1e-12


def test_noise_independence(orc):
    z = orc.noise(11, 5, NS)
    lim = 5 / np.sqrt(NS)
    for lag in (1, 2, 3, 1024):                                                  # lag 1 pairs the two draws of one Philox block
        for a, b in ((z.real, z.real), (z.imag, z.imag), (z.real, z.imag)):
            assert abs(np.mean(a[:-lag] * b[lag:])) < lim
    for other in (orc.noise(11, 6, NS), orc.noise(12, 5, NS), orc.noise(11 + (1 << 32), 5, NS), orc.noise(11, 5 + (1 << 32), NS)):
        assert abs(np.mean(z.real * other.real)) < lim and abs(np.mean(z.imag * other.imag)) < lim
        assert abs(np.vdot(z, other)) / NS < 2 * lim
    # squares too (a shared radius would pass the linear test)
    assert abs(np.corrcoef(np.abs(z[0::2]) ** 2, np.abs(z[1::2]) ** 2)[0, 1]) < lim * 2


def test_noise_addressing(orc):
    z = orc.noise(3, 1, 4096)
    assert np.array_equal(orc.noise(3, 1, 100, first=37), z[37:137])            # a window is a window, odd start included
    assert np.array_equal(orc.noise(3, 1, 1, first=4095), z[4095:])
    hi = orc.noise(3, 1, 64, first=1 << 33)                                      # block index 2^32: the second counter word
    assert np.abs(hi - z[:64]).min() > 0
    straddle = orc.noise(3, 1, 8, first=(1 << 33) - 4)
    assert np.array_equal(straddle[4:], hi[:4]) and np.abs(straddle[:4] - z[:4]).min() > 0


def _philox_inverse(out, key):
    """Invert the ten rounds with modular inverses of the two multipliers (written here, independently of the oracle)."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    inv0, inv1 = pow(M0, -1, 1 << 32), pow(M1, -1, 1 << 32)
    o = [int(v) for v in out]
    for r in reversed(range(10)):
        k0, k1 = (key[0] + r * W0) & 0xFFFFFFFF, (key[1] + r * W1) & 0xFFFFFFFF
        c2 = (o[1] * inv1) & 0xFFFFFFFF
        c0 = (o[3] * inv0) & 0xFFFFFFFF
        c1 = o[0] ^ ((M1 * c2) >> 32) ^ k0
        c3 = o[2] ^ ((M0 * c0) >> 32) ^ k1
        o = [c0, c1, c2, c3]
    return o


def test_philox_is_a_keyed_bijection_with_avalanche(orc):
    rng = np.random.default_rng(5)
    ctr = rng.integers(0, 1 << 32, size=(64, 4), dtype=np.uint64).astype(np.uint32)
    key = (0x243F6A88, 0x85A308D3)
    out = orc.philox4x32_10(ctr, key)
    for c, o in zip(ctr, out):
        assert _philox_inverse(o, key) == [int(v) for v in c]
    # flipping any single counter or key bit flips about half of the 128 output bits
    bits = lambda a: np.unpackbits(np.ascontiguousarray(a).view(np.uint8), axis=-1)
    base = bits(out)
    for word in range(4):
        for bit in (0, 7, 16, 31):
            c2 = ctr.copy()
            c2[:, word] ^= np.uint32(1 << bit)
            frac = np.mean(bits(orc.philox4x32_10(c2, key)) != base)
            assert 0.45 < frac < 0.55, (word, bit, frac)
    for kw in range(2):
        k2 = list(key)
        k2[kw] ^= 1 << 13
        frac = np.mean(bits(orc.philox4x32_10(ctr, tuple(k2))) != base)
        assert 0.45 < frac < 0.55
    # uniform bytes: chi-square over the 256 byte values of 2^18 output words
    big = orc.philox4x32_10(np.stack([np.arange(1 << 16, dtype=np.uint32)] + [np.zeros(1 << 16, np.uint32)] * 3, axis=1), key)
    cnt = np.bincount(big.view(np.uint8).ravel(), minlength=256)
    assert stats.chisquare(cnt).pvalue > 1e-3


def philox_kat_vectors():
    """(counter[4], key[2], expected[4]) from tests/golden/philox_kat.txt (Salmon et al., SC'11; Random123)."""
    out = []
    with open(os.path.join(GOLDEN, "philox_kat.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].replace("->", " ").split()
            if line:
                w = [int(x, 16) for x in line]
                assert len(w) == 10
                out.append((w[0:4], w[4:6], w[6:10]))
    assert len(out) == 3
    return out


def test_philox_known_answer_vectors(orc):
    """The name "Philox-4x32-10" is a claim the published algorithm fixes: the three known-answer vectors of its authors
    (all-zero, all-ones, pi digits) must come out word for word."""
    for ctr, key, want in philox_kat_vectors():
        got = orc.philox4x32_10(np.array([ctr], dtype=np.uint32), key)[0]
        assert [int(v) for v in got] == want, ([hex(int(v)) for v in got], [hex(v) for v in want])
    # vectorised over counters: the same three in one call per key
    for ctr, key, want in philox_kat_vectors():
        many = np.array([ctr, [1, 2, 3, 4], ctr], dtype=np.uint32)
        got = orc.philox4x32_10(many, key)
        assert [int(v) for v in got[0]] == want and [int(v) for v in got[2]] == want
    # and noise() addresses the blocks as DESIGN.md Q29 says: block i of (seed, stream) = counter (i lo, i hi, stream lo,
    # stream hi), key (seed lo, seed hi); draw 2i from (x0, x1), draw 2i+1 from (x2, x3), 23-bit uniforms
    ctr, key, want = philox_kat_vectors()[2]
    i = ctr[0] | (ctr[1] << 32)
    stream = ctr[2] | (ctr[3] << 32)
    seed = key[0] | (key[1] << 32)
    z = orc.noise(seed, stream, 2, first=2 * i)
    for d in range(2):
        u = ((want[2 * d] >> 9) + 0.5) / 2.0 ** 23
        f = ((want[2 * d + 1] >> 9) + 0.5) / 2.0 ** 23
        ref = np.sqrt(-2.0 * np.log(u)) * np.exp(2j * np.pi * f)
        assert abs(z[d] - ref) < 1e-14 * abs(ref)
