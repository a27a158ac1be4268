"""ctypes wrapper around oracle/orc.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never imports the product package.

`build()` compiles orc.c with gcc into oracle/liborc.so (a few seconds); every
wrapper below only marshals numpy arrays into the C calls declared in orc.h.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liborc.so")
_SRC = os.path.join(_HERE, "orc.c")
_HDR = os.path.join(_HERE, "orc.h")

PSD_KOLMOGOROV, PSD_VON_KARMAN, PSD_OCEAN_NIKISHOV, PSD_POWER_LAW = 0, 1, 2, 3
H_FRESNEL, H_ANGULAR_SPECTRUM = 0, 1


class _Psd(C.Structure):
    _fields_ = [("kind", C.c_int), ("L0", C.c_double), ("l0", C.c_double),
                ("km_coeff", C.c_double), ("chi_T", C.c_double), ("eps", C.c_double),
                ("w", C.c_double), ("eta", C.c_double), ("alpha", C.c_double), ("A", C.c_double)]


class _Stats(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("power", "cx", "cy", "sxx", "syy", "sxy", "w2",
                                           "I_axis", "roi_sumI", "roi_sumI2")] + \
               [("roi_n", C.c_longlong)]


@dataclass
class Psd:
    kind: int = PSD_KOLMOGOROV
    L0: float = 0.0
    l0: float = 0.0
    km_coeff: float = 0.0
    chi_T: float = 0.0
    eps: float = 0.0
    w: float = 0.0
    eta: float = 0.0
    alpha: float = 0.0
    A: float = 0.0

    def c(self) -> _Psd:
        return _Psd(self.kind, self.L0, self.l0, self.km_coeff, self.chi_T, self.eps, self.w, self.eta,
                    self.alpha, self.A)


def build(force: bool = False) -> str:
    """Compile the oracle (gcc -O2, strict IEEE: no -ffast-math)."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < newest:
        tmp = _SO + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_psd_f.restype = C.c_double
        _lib.orc_r0.restype = C.c_double
    return _lib


def _p(a, ty=C.c_double):
    return a.ctypes.data_as(C.POINTER(ty)) if a is not None else None


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed rc={rc}")


# ---- P0 ---------------------------------------------------------------------
def fft1d(a, sign=-1):
    a = _c128(a).copy()
    _chk(lib().orc_fft1d(_p(a), C.c_int(a.shape[-1]), C.c_int(sign)), "fft1d")
    return a


def dft1d_naive(a, sign=-1):
    a = _c128(a).copy()
    _chk(lib().orc_dft1d_naive(_p(a), C.c_int(a.shape[-1]), C.c_int(sign)), "dft1d_naive")
    return a


def fft2d(a, sign=-1):
    a = _c128(a).copy()
    assert a.ndim == 2 and a.shape[0] == a.shape[1]
    _chk(lib().orc_fft2d(_p(a), C.c_int(a.shape[0]), C.c_int(sign)), "fft2d")
    return a


# ---- O2 ---------------------------------------------------------------------
def r0(lam, cn2, dz):
    return lib().orc_r0(C.c_double(lam), C.c_double(cn2), C.c_double(dz))


def psd_f(psd: Psd, lam, cn2, dz, f):
    pc = psd.c()
    fn = lib().orc_psd_f
    f = np.atleast_1d(np.asarray(f, dtype=np.float64))
    out = np.array([fn(C.byref(pc), C.c_double(lam), C.c_double(cn2), C.c_double(dz), C.c_double(x))
                    for x in f.ravel()])
    return out.reshape(f.shape)


# ---- O3-O5 ------------------------------------------------------------------
def make_screens(N, dx, psd: Psd, lam, cn2, dz, n_sh, noise, noise_sh, keep_spectrum=True):
    """noise: float32 [B][S][N][N][2]; noise_sh: float32 [B][S][n_sh][3][3][2] (or None).
    Returns (screens f64 [B][S][N][N], spectrum c128 or None, sh_coef c128 or None)."""
    noise = _f32(noise)
    B, S = noise.shape[0], noise.shape[1]
    cn2, dz = _f64(cn2), _f64(dz)
    assert cn2.shape == (S,) and dz.shape == (S,)
    screens = np.empty((B, S, N, N), dtype=np.float64)
    spectrum = np.empty((B, S, N, N), dtype=np.complex128) if keep_spectrum else None
    sh = np.zeros((B, S, max(n_sh, 1), 3, 3), dtype=np.complex128) if n_sh > 0 else None
    nsh = _f32(noise_sh) if n_sh > 0 else None
    pc = psd.c()
    _chk(lib().orc_make_screens(C.c_int(N), C.c_double(dx), C.byref(pc), C.c_double(lam),
                                C.c_int(B), C.c_int(S), _p(cn2), _p(dz), C.c_int(n_sh),
                                _p(noise, C.c_float), _p(nsh, C.c_float),
                                _p(spectrum), _p(sh), _p(screens)), "make_screens")
    return screens, spectrum, sh


def synthesize(N, dx, n_sh, spectrum, sh_coef, part="re"):
    """Screens from stored spectra / subharmonic coefficients: the real part of the synthesis (the paper's screen,
    Q3) or, with part="im", its imaginary part -- a second screen of the same statistics from the same noise."""
    spectrum = _c128(spectrum)
    B, S = spectrum.shape[0], spectrum.shape[1]
    sh = _c128(sh_coef) if n_sh > 0 else None
    screens = np.empty((B, S, N, N), dtype=np.float64)
    fn = lib().orc_synthesize_im if part == "im" else lib().orc_synthesize
    _chk(fn(C.c_int(N), C.c_double(dx), C.c_int(B), C.c_int(S), C.c_int(n_sh),
            _p(spectrum), _p(sh), _p(screens)), "synthesize")
    return screens


def evolve_screens(N, dx, psd: Psd, lam, cn2, dz, n_sh, a, vx, vy, T, fresh, fresh_sh,
                   spectrum, sh_coef):
    """Updates spectrum / sh_coef IN PLACE (must be contiguous c128) and returns the screens."""
    fresh = _f32(fresh)
    B, S = fresh.shape[0], fresh.shape[1]
    assert spectrum.dtype == np.complex128 and spectrum.flags.c_contiguous
    cn2, dz = _f64(cn2), _f64(dz)
    screens = np.empty((B, S, N, N), dtype=np.float64)
    fsh = _f32(fresh_sh) if n_sh > 0 else None
    if n_sh > 0:
        assert sh_coef.dtype == np.complex128 and sh_coef.flags.c_contiguous
    pc = psd.c()
    _chk(lib().orc_evolve_screens(C.c_int(N), C.c_double(dx), C.byref(pc), C.c_double(lam),
                                  C.c_int(B), C.c_int(S), _p(cn2), _p(dz), C.c_int(n_sh),
                                  C.c_double(a), C.c_double(vx), C.c_double(vy), C.c_double(T),
                                  _p(fresh, C.c_float), _p(fsh, C.c_float),
                                  _p(spectrum), _p(sh_coef) if n_sh > 0 else None, _p(screens)),
         "evolve_screens")
    return screens


# ---- O6-O7 ------------------------------------------------------------------
def _screen_args(screens, B, N, shared):
    if screens is None:
        return None, 0, 0
    screens = _f64(screens)
    if shared:
        assert screens.ndim == 3
        return screens, 0, screens.shape[0]
    assert screens.ndim == 4 and screens.shape[0] == B
    return screens, screens.shape[1] * N * N, screens.shape[1]


def propagate(N, dx, lam, dz, field, screens=None, shared_screens=False, win_order=0,
              win_sigma_frac=0.47, n0=1.0, h_kind=H_FRESNEL, return_planes=False):
    field = _c128(field)
    B = field.shape[0]
    dz = _f64(dz)
    n_steps = dz.shape[0]
    scr, stride, S = _screen_args(screens, B, N, shared_screens)
    out = np.empty_like(field)
    planes = np.empty((B, n_steps, N, N), dtype=np.complex128) if return_planes else None
    _chk(lib().orc_propagate(C.c_int(N), C.c_double(dx), C.c_double(lam), C.c_double(n0),
                             C.c_int(B), C.c_int(n_steps), _p(dz), _p(scr), C.c_longlong(stride),
                             C.c_int(S), C.c_int(win_order), C.c_double(win_sigma_frac),
                             C.c_int(h_kind), _p(field), _p(out), _p(planes)), "propagate")
    return (out, planes) if return_planes else out


def propagate_adjoint(N, dx, lam, dz, g_out, screens=None, shared_screens=False, win_order=0,
                      win_sigma_frac=0.47, n0=1.0, h_kind=H_FRESNEL, planes=None):
    g_out = _c128(g_out)
    B = g_out.shape[0]
    dz = _f64(dz)
    n_steps = dz.shape[0]
    scr, stride, S = _screen_args(screens, B, N, shared_screens)
    g_in = np.empty_like(g_out)
    grad = None
    if planes is not None:
        planes = _c128(planes)
        assert planes.shape == (B, n_steps, N, N)
        grad = np.zeros((B, max(S, 1), N, N), dtype=np.float64)
    _chk(lib().orc_propagate_adjoint(C.c_int(N), C.c_double(dx), C.c_double(lam), C.c_double(n0),
                                     C.c_int(B), C.c_int(n_steps), _p(dz), _p(scr),
                                     C.c_longlong(stride), C.c_int(S), C.c_int(win_order),
                                     C.c_double(win_sigma_frac), C.c_int(h_kind),
                                     _p(g_out), _p(g_in), _p(planes), _p(grad)), "propagate_adjoint")
    return (g_in, grad) if planes is not None else g_in


# ---- O8 ---------------------------------------------------------------------
STAT_FIELDS = ("power", "cx", "cy", "sxx", "syy", "sxy", "w2", "I_axis", "roi_sumI", "roi_sumI2", "roi_n")


def beam_stats(N, dx, field, roi_frac=0.5):
    field = _c128(field)
    B = field.shape[0]
    arr = (_Stats * B)()
    _chk(lib().orc_beam_stats(C.c_int(N), C.c_double(dx), C.c_int(B), _p(field),
                              C.c_double(roi_frac), arr), "beam_stats")
    return [{k: getattr(arr[b], k) for k in STAT_FIELDS} for b in range(B)]


def welford(N, field, mean, M2, count):
    """mean / M2: float64 [N][N] updated in place; returns the new count."""
    field = _c128(field)
    cnt = C.c_longlong(count)
    _chk(lib().orc_welford(C.c_int(N), C.c_int(field.shape[0]), _p(field), _p(mean), _p(M2),
                           C.byref(cnt)), "welford")
    return cnt.value


# ---- O9 ---------------------------------------------------------------------
def phase_mul(N, theta, field, sign=1.0):
    field = _c128(field)
    theta = _f64(theta)
    out = np.empty_like(field)
    _chk(lib().orc_phase_mul(C.c_int(N), C.c_int(field.shape[0]), _p(theta), C.c_double(sign),
                             _p(field), _p(out)), "phase_mul")
    return out


def dft2_centered(N, field, inverse=False):
    field = _c128(field)
    out = np.empty_like(field)
    _chk(lib().orc_dft2_centered(C.c_int(N), C.c_int(field.shape[0]), C.c_int(int(inverse)),
                                 _p(field), _p(out)), "dft2_centered")
    return out


def aperture(N, dx, radius, field):
    """Circular aperture of `radius` metres; the integer threshold floor((radius/dx)^2) is taken here in double."""
    field = _c128(field)
    out = np.empty_like(field)
    r2 = int(np.floor((radius / dx) ** 2))
    _chk(lib().orc_aperture(C.c_int(N), C.c_int(field.shape[0]), C.c_longlong(r2), _p(field), _p(out)), "aperture")
    return out


def phase_grad(N, g, u):
    g, u = _c128(g), _c128(u)
    out = np.empty(g.shape, dtype=np.float64)
    _chk(lib().orc_phase_grad(C.c_int(N), C.c_int(g.shape[0]), _p(g), _p(u), _p(out)), "phase_grad")
    return out


def adam_step(grad, lr, t, m, v, theta, beta1=0.9, beta2=0.999, eps=1e-8):
    """Adam (Kingma & Ba), the optimiser of PAPER.md:115, on a mask shared by the batch: g = mean_b grad[b].
    Returns new (m, v, theta) in float64."""
    g = np.mean(np.asarray(grad, dtype=np.float64), axis=0)
    m = beta1 * np.asarray(m, dtype=np.float64) + (1.0 - beta1) * g
    v = beta2 * np.asarray(v, dtype=np.float64) + (1.0 - beta2) * g * g
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    return m, v, np.asarray(theta, dtype=np.float64) - lr * mhat / (np.sqrt(vhat) + eps)


# ---- path description (PAPER.md:393 S21, :375 S18, :380 S19) ------------------------------------------------
def hv57_cn2(h, A, V=21.0, ground_scale=1000.0):
    """Hufnagel-Valley 5/7 as printed in S21 (third scale height 1000 m there; the textbook value is 100 m)."""
    h = np.asarray(h, dtype=np.float64)
    return (0.00594 * (V / 27.0) ** 2 * (1e-5 * h) ** 10 * np.exp(-h / 1000.0) + 2.7e-16 * np.exp(-h / 1500.0)
            + A * np.exp(-h / ground_scale))


def hv57_slab_integral(a, b, A, V=21.0, ground_scale=1000.0):
    """int_a^b Cn2(h) dh in closed form: exponentials, and the h^10 exp(-h/1000) term through the regularised
    incomplete gamma function."""
    from scipy import special
    e = lambda s: s * (np.exp(-a / s) - np.exp(-b / s))
    g11 = special.gamma(11.0) * (special.gammainc(11.0, b / 1000.0) - special.gammainc(11.0, a / 1000.0))
    return 0.00594 * (V / 27.0) ** 2 * 1e-50 * 1000.0 ** 11 * g11 + 2.7e-16 * e(1500.0) + A * e(ground_scale)


def hv57_path(h0, L, n, lam, A, V=21.0, ground_scale=1000.0):
    """Equal slabs: (cn2[n] slab means, dz[n], Rytov variance by S19 with adaptive quadrature, r0 by S18)."""
    from scipy import integrate
    k = 2.0 * np.pi / lam
    edges = h0 + L * np.arange(n + 1) / n
    ints = np.array([hv57_slab_integral(edges[j], edges[j + 1], A, V, ground_scale) for j in range(n)])
    w = integrate.quad(lambda z: float(hv57_cn2(h0 + z, A, V, ground_scale)) * (1.0 - z / L) ** (5.0 / 3.0), 0.0, L,
                       epsabs=0, epsrel=1e-12, limit=400)[0]
    rytov = 3.27 * k ** (7.0 / 6.0) * L ** (5.0 / 6.0) * w
    return ints / (L / n), np.full(n, L / n), rytov, (0.423 * k * k * ints.sum()) ** (-3.0 / 5.0)


# ---- screen placement (Sec 2.4; Eq. 7 with reading Q17; steps of :109 with reading Q28) -------
def dz_max_angular_spectrum(N, dx, lam, n0=1.0):
    """Largest step the angular-spectrum H (Eq. 6) supports before its phase aliases on the grid.
    Phase psi = dz sqrt(n0^2 k0^2 - kappa^2); |d psi / d kappa| dkappa <= pi at the largest axis frequency
    kappa0 = pi / dx with dkappa = 2 pi / (N dx) gives dz <= (N dx / 2) sqrt(n0^2 k0^2 - kappa0^2) / kappa0 (Q17:
    Eq. 7 as printed has the ratio inverted and kappa0 = 2 pi / dx).  Paraxial limit: N dx^2 n0 / lam."""
    k0 = 2.0 * np.pi / lam
    kap = np.pi / dx
    if n0 * k0 <= kap:
        return 0.0
    return 0.5 * N * dx * np.sqrt(n0 * n0 * k0 * k0 - kap * kap) / kap


def interval_rytov(cn2_of_z, a, b, lam, kinks=()):
    """S19 over the interval [a, b], z measured from a; adaptive quadrature, piece by piece between
    the profile's kinks."""
    from scipy import integrate
    k = 2.0 * np.pi / lam
    d = b - a
    if d <= 0:
        return 0.0
    cuts = [a] + [float(p) for p in kinks if a < p < b] + [b]
    w = sum(integrate.quad(lambda z: float(cn2_of_z(z)) * (1.0 - (z - a) / d) ** (5.0 / 3.0), lo, hi,
                           epsabs=0, epsrel=1e-13)[0] for lo, hi in zip(cuts[:-1], cuts[1:]))
    return 3.27 * k ** (7.0 / 6.0) * d ** (5.0 / 6.0) * w


def place_screens(z_prof, cn2_prof, edges, lam, rytov_limit, dz_max=0.0, return_stages=False):
    """The placement routine of PAPER.md:109, sentence by sentence, on a piecewise-linear Cn2(z) profile:
      1. an interval whose Rytov variance exceeds the limit is halved until every piece is within it;
      2. neighbours whose union stays within the limit are merged (left to right);
      3. "linear fit": marching from the start, each interval's end is moved to where the straight line through
         (last old edge within the limit, its variance) and (next old edge, its variance) meets the limit (Q28);
         if the profile is not convex enough for that point to be within the limit, the move is halved until it is;
      4. an interval longer than dz_max (Eq. 7) is halved until it is not.
    Returns dz[n], the slab-mean cn2[n] and the interval Rytov variances."""
    from scipy import integrate
    z_prof = np.asarray(z_prof, dtype=np.float64)
    cn2_prof = np.asarray(cn2_prof, dtype=np.float64)
    f = lambda z: np.interp(z, z_prof, cn2_prof)
    ry = lambda a, b: interval_rytov(f, a, b, lam, z_prof)
    e = [float(x) for x in edges]
    # 1
    out = [e[0]]
    for a, b in zip(e[:-1], e[1:]):
        parts = 1
        while max(ry(a + (b - a) * i / parts, a + (b - a) * (i + 1) / parts) for i in range(parts)) > rytov_limit:
            parts *= 2
        out += [a + (b - a) * (i + 1) / parts for i in range(parts)]
    s1_edges = list(out)
    # 2
    i = 0
    while i + 2 < len(out):
        if ry(out[i], out[i + 2]) <= rytov_limit:
            del out[i + 1]
        else:
            i += 1
    s2_edges = list(out)
    # 3
    new, a, j, end = [out[0]], out[0], 1, out[-1]
    while True:
        b1, v1 = a, 0.0
        while j < len(out) and (out[j] <= a or ry(a, out[j]) <= rytov_limit):
            if out[j] > a:
                b1, v1 = out[j], ry(a, out[j])
            j += 1
        if j >= len(out):
            if end > a:
                new.append(end)
            break
        b2, v2 = out[j], ry(a, out[j])
        step = (rytov_limit - v1) / (v2 - v1) * (b2 - b1)
        while ry(a, b1 + step) > rytov_limit:
            step *= 0.5
        new.append(b1 + step)
        a = b1 + step
    s3_edges = list(new)
    # 4
    fin = [new[0]]
    for a, b in zip(new[:-1], new[1:]):
        parts = 1
        while dz_max > 0 and (b - a) / parts > dz_max:
            parts *= 2
        fin += [a + (b - a) * (i + 1) / parts for i in range(parts)]
    fin = np.array(fin)
    dz = np.diff(fin)
    def seg(a, b):
        cuts = [a] + [float(p) for p in z_prof if a < p < b] + [b]
        return sum(integrate.quad(lambda z: float(f(z)), lo, hi, epsabs=0, epsrel=1e-13)[0]
                   for lo, hi in zip(cuts[:-1], cuts[1:]))
    cn2 = np.array([seg(a, b) for a, b in zip(fin[:-1], fin[1:])]) / dz
    rys = np.array([ry(a, b) for a, b in zip(fin[:-1], fin[1:])])
    if return_stages:
        return dz, cn2, rys, dict(split=np.array(s1_edges), merged=np.array(s2_edges), fitted=np.array(s3_edges))
    return dz, cn2, rys


# ---- counter-based noise (the "unit-variance complex Gaussian" draws of S16; reading Q29) -------------
def philox4x32_10(counter, key):
    """Philox-4x32 with 10 rounds (Salmon et al., SC'11), vectorised over counters.
    counter: uint32 [n][4], key: (k0, k1).  Returns uint32 [n][4].
    One round:  (c0, c1, c2, c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)),
    then the key is bumped by the Weyl constants."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    c = [np.asarray(counter)[:, i].astype(np.uint64) for i in range(4)]
    k0, k1 = int(key[0]) & 0xFFFFFFFF, int(key[1]) & 0xFFFFFFFF
    mask = np.uint64(0xFFFFFFFF)
    for _ in range(10):
        p0 = np.uint64(M0) * c[0]
        p1 = np.uint64(M1) * c[2]
        c = [(p1 >> np.uint64(32)) ^ c[1] ^ np.uint64(k0), p1 & mask,
             (p0 >> np.uint64(32)) ^ c[3] ^ np.uint64(k1), p0 & mask]
        k0 = (k0 + W0) & 0xFFFFFFFF
        k1 = (k1 + W1) & 0xFFFFFFFF
    return np.stack(c, axis=1).astype(np.uint32)


def noise(seed, stream, n, first=0):
    """n complex draws, Re and Im each N(0, 1) (Q3), numbered first .. first+n-1 within (seed, stream).
    Draws 2i and 2i+1 come from the Philox block with counter (i mod 2^32, i >> 32, stream mod 2^32, stream >> 32) and
    key (seed mod 2^32, seed >> 32): words (x0, x1) make draw 2i, (x2, x3) draw 2i+1, by Box-Muller on 23-bit
    uniforms (k + 1/2 with k < 2^23 is exact in fp32 and fp64):  u = ((x_even >> 9) + 1/2) 2^-23,  f = ((x_odd >> 9) + 1/2) 2^-23,
    z = sqrt(-2 ln u) (cos 2 pi f + i sin 2 pi f)."""
    i0, i1 = first // 2, (first + n + 1) // 2
    idx = np.arange(i0, i1, dtype=np.uint64)
    ctr = np.stack([idx & np.uint64(0xFFFFFFFF), idx >> np.uint64(32),
                    np.full(idx.shape, int(stream) & 0xFFFFFFFF, dtype=np.uint64),
                    np.full(idx.shape, (int(stream) >> 32) & 0xFFFFFFFF, dtype=np.uint64)], axis=1)
    x = philox4x32_10(ctr, (int(seed) & 0xFFFFFFFF, (int(seed) >> 32) & 0xFFFFFFFF)).astype(np.float64)
    x = x.reshape(-1, 2)                                                   # one (radius word, angle word) pair per draw
    u = (np.floor(x[:, 0] / 512.0) + 0.5) / 8388608.0
    f = (np.floor(x[:, 1] / 512.0) + 0.5) / 8388608.0
    z = np.sqrt(-2.0 * np.log(u)) * np.exp(2j * np.pi * f)
    return z[first - 2 * i0: first - 2 * i0 + n]
