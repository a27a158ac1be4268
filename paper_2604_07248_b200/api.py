"""Thin ctypes binding of include/ssp.h -- argument marshalling only.

Every function below has the name of the C entry point it calls (minus the `ssp_` prefix) and
does nothing but turn torch CUDA tensors into device pointers, python lists into host arrays
and return codes into exceptions.  All arithmetic of the method runs in the library's kernels.
PyTorch is used for device memory and streams only.  There is no CPU fallback: a missing
libssp.so, a missing GPU or a non-CUDA tensor raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libssp.so")

PSD_KOLMOGOROV, PSD_VON_KARMAN, PSD_OCEAN_NIKISHOV, PSD_POWER_LAW = 0, 1, 2, 3
H_FRESNEL, H_ANGULAR_SPECTRUM = 0, 1
OK, EINVAL, EUNSUPPORTED, EWORKSPACE, ECUDA = 0, -1, -2, -3, -4

# every symbol include/ssp.h declares (tests/test_abi.py checks the header against this list)
SYMBOLS = (
    "ssp_create", "ssp_destroy", "ssp_last_error", "ssp_version", "ssp_launch_count",
    "ssp_workspace_bytes", "ssp_make_screens", "ssp_evolve_screens", "ssp_evolve_screens_seeded", "ssp_make_screens_seeded", "ssp_make_screens_pair", "ssp_evolve_screens_pair", "ssp_propagate",
    "ssp_propagate_adjoint", "ssp_beam_stats", "ssp_beam_stats_static", "ssp_propagate_host", "ssp_phase_mul",
    "ssp_dft2_centered", "ssp_phase_grad", "ssp_inner_products", "ssp_lincomb", "ssp_aperture", "ssp_adam_update", "ssp_hv57_cn2", "ssp_hv57_path", "ssp_dz_max", "ssp_place_screens", "ssp_fill_noise", "ssp_philox_words", "ssp_evolve_propagate", "ssp_mae_loss", "ssp_frame_chunk", "ssp_frame_host",
    "ssp_profile_enable", "ssp_profile_report",
)


class SspError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ssp error {code}: {msg}")
        self.code = code


class Grid(C.Structure):
    _fields_ = [("N", C.c_int), ("dx", C.c_double)]


class Psd(C.Structure):
    _fields_ = [("kind", C.c_int), ("L0", C.c_double), ("l0", C.c_double), ("km_coeff", C.c_double),
                ("chi_T", C.c_double), ("eps", C.c_double), ("w", C.c_double), ("eta", C.c_double),
                ("alpha", C.c_double), ("A", C.c_double)]


class Hv57(C.Structure):
    _fields_ = [("A", C.c_double), ("V", C.c_double), ("ground_scale", C.c_double)]


class Window(C.Structure):
    _fields_ = [("order", C.c_int), ("sigma_frac", C.c_double)]


class Ar(C.Structure):
    _fields_ = [("a", C.c_double), ("vx", C.c_double), ("vy", C.c_double), ("T", C.c_double),
                ("seed", C.c_ulonglong), ("frame", C.c_ulonglong)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("power", "cx", "cy", "sxx", "syy", "sxy", "w2", "I_axis",
                                           "roi_sumI", "roi_sumI2")] + [("roi_n", C.c_longlong)]


STATS_BYTES = C.sizeof(Stats)
STAT_FIELDS = tuple(n for n, _ in Stats._fields_)
STATS_STATIC_MAX_FIELDS = 1024     # SSP_STATS_STATIC_MAX_FIELDS of include/ssp.h

_lib = None


def load():
    """dlopen libssp.so (built in-tree by paper_2604_07248_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2604_07248_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.ssp_last_error.restype = C.c_char_p
    lib.ssp_last_error.argtypes = [C.c_void_p]
    lib.ssp_version.restype = C.c_char_p
    lib.ssp_launch_count.restype = C.c_longlong
    lib.ssp_launch_count.argtypes = [C.c_void_p]
    lib.ssp_workspace_bytes.restype = C.c_size_t
    lib.ssp_workspace_bytes.argtypes = [Grid, C.c_int, C.c_int]
    lib.ssp_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p]
    lib.ssp_destroy.argtypes = [C.c_void_p]
    P, D, I, L = C.c_void_p, C.c_double, C.c_int, C.c_longlong
    lib.ssp_make_screens.argtypes = [P, Grid, C.POINTER(Psd), D, I, I, P, P, I, P, P, P, P, P, P, C.c_size_t]
    lib.ssp_make_screens_pair.argtypes = [P, Grid, C.POINTER(Psd), D, I, I, P, P, I, P, P, P, P, P, P, P, C.c_size_t]
    lib.ssp_evolve_screens_pair.argtypes = [P, Grid, C.POINTER(Psd), D, I, I, P, P, I, D, D, D, D, P, P, P, P, P, P, P,
                                            C.c_size_t]
    lib.ssp_evolve_screens.argtypes = [P, Grid, C.POINTER(Psd), D, I, I, P, P, I, D, D, D, D, P, P, P, P, P, P,
                                       C.c_size_t]
    lib.ssp_make_screens_seeded.argtypes = [P, Grid, C.POINTER(Psd), D, I, I, P, P, I, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong,
                                            P, P, P, P, P, C.c_size_t]
    lib.ssp_evolve_screens_seeded.argtypes = [P, Grid, C.POINTER(Psd), D, I, I, P, P, I, D, D, D, D, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, P, P, P, P, P,
                                              C.c_size_t]
    lib.ssp_propagate.argtypes = [P, Grid, D, D, I, I, I, P, P, L, I, Window, P, P, P, P, D, P, C.c_size_t]
    lib.ssp_evolve_propagate.argtypes = [P, Grid, C.POINTER(Psd), D, D, I, I, P, P, I, D, D, D, D, P, P, P, P, Window, P, P,
                                         P, D, P, P, C.c_size_t]
    lib.ssp_propagate_adjoint.argtypes = [P, Grid, D, D, I, I, I, P, P, L, I, Window, P, P, P, P, P, C.c_size_t]
    lib.ssp_beam_stats.argtypes = [P, Grid, I, P, D, P, P, P, C.POINTER(L)]
    lib.ssp_beam_stats_static.argtypes = [P, Grid, I, P, D, P]
    lib.ssp_propagate_host.argtypes = [P, Grid, D, D, I, I, I, P, P, L, I, Window, P, P, P, D, P, P, P, P,
                                       C.c_size_t]
    lib.ssp_frame_chunk.argtypes = [I]
    lib.ssp_frame_host.argtypes = [P, Grid, P, D, D, I, I, I, P, P, I, P, Window, P, P, P, D, P, P, P, P, P, P, P, P,
                                   C.c_size_t, P, P]
    lib.ssp_phase_mul.argtypes = [P, Grid, I, P, D, P, P]
    lib.ssp_dft2_centered.argtypes = [P, Grid, I, I, P, P, P, C.c_size_t]
    lib.ssp_phase_grad.argtypes = [P, Grid, I, P, P, P]
    lib.ssp_aperture.argtypes = [P, Grid, I, D, P, P]
    lib.ssp_hv57_cn2.argtypes = [C.POINTER(Hv57), D]
    lib.ssp_hv57_cn2.restype = D
    lib.ssp_hv57_path.argtypes = [C.POINTER(Hv57), D, D, I, D, P, P, P, P]
    lib.ssp_fill_noise.argtypes = [P, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, P]
    lib.ssp_philox_words.argtypes = [P, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, C.c_ulonglong, P]
    lib.ssp_dz_max.argtypes = [Grid, D, D]
    lib.ssp_dz_max.restype = D
    lib.ssp_place_screens.argtypes = [P, P, I, P, I, D, D, D, I, P, P, P, P]
    lib.ssp_adam_update.argtypes = [P, Grid, I, P, D, D, D, D, I, P, P, P]
    lib.ssp_inner_products.argtypes = [P, Grid, I, P, P, P]
    lib.ssp_mae_loss.argtypes = [P, Grid, I, P, P, P, P]
    lib.ssp_lincomb.argtypes = [P, Grid, I, P, P, P, P, P]
    lib.ssp_profile_enable.argtypes = [P, I]
    lib.ssp_profile_report.argtypes = [P, C.c_char_p, C.c_size_t]
    _lib = lib
    return lib


def version() -> str:
    return load().ssp_version().decode()


def workspace_bytes(N: int, dx: float, B: int, S: int) -> int:
    return int(load().ssp_workspace_bytes(Grid(N, dx), B, S))


def _dev(t: Optional[torch.Tensor], dtype=None):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda:
        raise TypeError("ssp: expected a CUDA tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError("ssp: tensor must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"ssp: expected {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _host_doubles(x: Sequence[float]):
    arr = (C.c_double * len(x))(*[float(v) for v in x])
    return arr


@dataclass
class PsdParams:
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

    def c(self) -> Psd:
        return Psd(self.kind, self.L0, self.l0, self.km_coeff, self.chi_T, self.eps, self.w, self.eta,
                   self.alpha, self.A)


def hv57_cn2(h, A, V=21.0, ground_scale=0.0):
    """Hufnagel-Valley 5/7 Cn2 at height h [m] (host call, no context needed)."""
    return load().ssp_hv57_cn2(C.byref(Hv57(A, V, ground_scale)), float(h))


def hv57_path(h0, L, n, lam, A, V=21.0, ground_scale=0.0):
    """Equal slabs of a vertical HV5/7 path: (cn2[n], dz[n], rytov variance, r0) as numpy / floats."""
    import numpy as np
    cn2, dz = np.empty(n), np.empty(n)
    ry, r0 = C.c_double(), C.c_double()
    rc = load().ssp_hv57_path(C.byref(Hv57(A, V, ground_scale)), float(h0), float(L), int(n), float(lam),
                              cn2.ctypes.data_as(C.c_void_p), dz.ctypes.data_as(C.c_void_p), C.byref(ry), C.byref(r0))
    if rc != OK:
        raise SspError(rc, "ssp_hv57_path: bad arguments")
    return cn2, dz, ry.value, r0.value


def frame_chunk(B):
    """Fields per pipeline chunk of frame_host / propagate_host."""
    return int(load().ssp_frame_chunk(int(B)))


def dz_max(N, dx, lam, n0=1.0):
    """Largest alias-free angular-spectrum step on the grid (host call)."""
    return load().ssp_dz_max(Grid(N, dx), float(lam), float(n0))


def place_screens(z_prof, cn2_prof, edges, lam, rytov_limit, dz_max=0.0, max_out=4096):
    """Screen placement on a piecewise-linear Cn2 profile: (dz[n], cn2[n], rytov[n]) as numpy (host call)."""
    import numpy as np
    zp = np.ascontiguousarray(z_prof, dtype=np.float64)
    cp = np.ascontiguousarray(cn2_prof, dtype=np.float64)
    ed = np.ascontiguousarray(edges, dtype=np.float64)
    if zp.shape != cp.shape or zp.ndim != 1 or ed.ndim != 1:
        raise SspError(EINVAL, "place_screens: z_prof / cn2_prof / edges must be 1-D, profile arrays of equal length")
    dz, cn2, ry = np.empty(max_out), np.empty(max_out), np.empty(max_out)
    n = C.c_int()
    vp = lambda a: a.ctypes.data_as(C.c_void_p)
    rc = load().ssp_place_screens(vp(zp), vp(cp), zp.size, vp(ed), ed.size, float(lam), float(rytov_limit),
                                  float(dz_max), int(max_out), vp(dz), vp(cn2), vp(ry), C.byref(n))
    if rc != OK:
        raise SspError(rc, "ssp_place_screens failed (needs at least %d intervals)" % n.value)
    return dz[:n.value].copy(), cn2[:n.value].copy(), ry[:n.value].copy()


class Context:
    """ssp_ctx bound to a device and a torch stream (default: the current stream)."""

    def __init__(self, device: int = 0, stream: Optional[torch.cuda.Stream] = None):
        self._lib = load()
        if not torch.cuda.is_available():
            raise RuntimeError("ssp: no CUDA device (there is no CPU fallback)")
        self.device = device
        self.stream = stream if stream is not None else torch.cuda.current_stream(device)
        h = C.c_void_p()
        rc = self._lib.ssp_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise SspError(rc, "ssp_create failed (no usable sm_100 device?)")
        self._h = h
        self._ws = None

    def close(self):
        if getattr(self, "_h", None):
            self._lib.ssp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc: int):
        if rc != 0:
            raise SspError(rc, self._lib.ssp_last_error(self._h).decode())

    def profile_enable(self, on: bool = True):
        self._chk(self._lib.ssp_profile_enable(self._h, int(on)))

    def profile_report(self) -> dict:
        """{kernel class: {"launches", "ms", "bytes"}} since the last report; synchronises the stream."""
        buf = C.create_string_buffer(1 << 16)
        self._chk(self._lib.ssp_profile_report(self._h, buf, len(buf)))
        out = {}
        for line in buf.value.decode().splitlines():
            name, n, ms, by = line.split()
            out[name] = {"launches": int(n), "ms": float(ms), "bytes": float(by)}
        return out

    def launch_count(self) -> int:
        return int(self._lib.ssp_launch_count(self._h))

    def workspace(self, N: int, dx: float, B: int, S: int) -> torch.Tensor:
        """A cached torch byte buffer of at least ssp_workspace_bytes."""
        need = max(workspace_bytes(N, dx, B, S), 256)
        if self._ws is None or self._ws.numel() < need:
            self._ws = torch.empty(need, dtype=torch.uint8, device=f"cuda:{self.device}")
        return self._ws

    # ---- screens ---------------------------------------------------------------------------
    def make_screens(self, N, dx, psd: PsdParams, lam, cn2, dz, n_sh, noise, noise_sh=None,
                     spectrum=None, sh_coef=None, screens=None, ws=None, screens_im=None):
        """noise: complex64 [B][S][N][N]; noise_sh: complex64 [B][S][n_sh][3][3]; returns screens fp32.
        screens_im (fp32 [B][S][N][N]): also write the imaginary part of each synthesis as a second screen."""
        B, S = noise.shape[0], noise.shape[1]
        if screens is None:
            screens = torch.empty((B, S, N, N), dtype=torch.float32, device=noise.device)
        ws = self.workspace(N, dx, B, S) if ws is None else ws
        pc = psd.c()
        if screens_im is not None:
            self._chk(self._lib.ssp_make_screens_pair(
                self._h, Grid(N, dx), C.byref(pc), lam, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh,
                _dev(noise, torch.complex64), _dev(noise_sh, torch.complex64) if n_sh > 0 else None,
                _dev(spectrum, torch.complex64), _dev(sh_coef, torch.complex64), _dev(screens, torch.float32),
                _dev(screens_im, torch.float32), _dev(ws), ws.numel()))
            return screens
        self._chk(self._lib.ssp_make_screens(
            self._h, Grid(N, dx), C.byref(pc), lam, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh,
            _dev(noise, torch.complex64), _dev(noise_sh, torch.complex64) if n_sh > 0 else None,
            _dev(spectrum, torch.complex64), _dev(sh_coef, torch.complex64), _dev(screens, torch.float32),
            _dev(ws), ws.numel()))
        return screens

    def evolve_screens(self, N, dx, psd: PsdParams, lam, cn2, dz, n_sh, a, vx, vy, T, fresh, fresh_sh,
                       spectrum, sh_coef, screens=None, ws=None, screens_im=None):
        B, S = fresh.shape[0], fresh.shape[1]
        if screens is None:
            screens = torch.empty((B, S, N, N), dtype=torch.float32, device=fresh.device)
        ws = self.workspace(N, dx, B, S) if ws is None else ws
        pc = psd.c()
        if screens_im is not None:
            self._chk(self._lib.ssp_evolve_screens_pair(
                self._h, Grid(N, dx), C.byref(pc), lam, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh,
                a, vx, vy, T, _dev(fresh, torch.complex64), _dev(fresh_sh, torch.complex64) if n_sh > 0 else None,
                _dev(spectrum, torch.complex64), _dev(sh_coef, torch.complex64) if n_sh > 0 else None,
                _dev(screens, torch.float32), _dev(screens_im, torch.float32), _dev(ws), ws.numel()))
            return screens
        self._chk(self._lib.ssp_evolve_screens(
            self._h, Grid(N, dx), C.byref(pc), lam, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh,
            a, vx, vy, T, _dev(fresh, torch.complex64), _dev(fresh_sh, torch.complex64) if n_sh > 0 else None,
            _dev(spectrum, torch.complex64), _dev(sh_coef, torch.complex64) if n_sh > 0 else None,
            _dev(screens, torch.float32), _dev(ws), ws.numel()))
        return screens

    def make_screens_seeded(self, N, dx, psd: PsdParams, lam, cn2, dz, n_sh, seed, stream, first, B, noise_sh=None,
                            spectrum=None, sh_coef=None, screens=None, ws=None):
        """make_screens with the grid noise drawn inside the generator (draw first + element index of stream (seed, stream));
        B stacks of len(cn2) screens; N >= 512."""
        S = len(cn2)
        dev = torch.device("cuda", self.device)
        if screens is None:
            screens = torch.empty((B, S, N, N), dtype=torch.float32, device=dev)
        ws = self.workspace(N, dx, B, S) if ws is None else ws
        pc = psd.c()
        self._chk(self._lib.ssp_make_screens_seeded(
            self._h, Grid(N, dx), C.byref(pc), lam, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh,
            int(seed), int(stream), int(first), _dev(noise_sh, torch.complex64) if n_sh > 0 else None,
            _dev(spectrum, torch.complex64), _dev(sh_coef, torch.complex64) if n_sh > 0 else None,
            _dev(screens, torch.float32), _dev(ws), ws.numel()))
        return screens

    def evolve_screens_seeded(self, N, dx, psd: PsdParams, lam, cn2, dz, n_sh, a, vx, vy, T, seed, stream, first,
                              fresh_sh, spectrum, sh_coef, screens=None, ws=None):
        """evolve_screens with the fresh grid noise drawn inside the generator (draw first + element index of stream
        (seed, stream)): equals fill_noise + evolve_screens bit for bit; N >= 512 (EUNSUPPORTED below)."""
        B, S = spectrum.shape[0], spectrum.shape[1]
        if screens is None:
            screens = torch.empty((B, S, N, N), dtype=torch.float32, device=spectrum.device)
        ws = self.workspace(N, dx, B, S) if ws is None else ws
        pc = psd.c()
        self._chk(self._lib.ssp_evolve_screens_seeded(
            self._h, Grid(N, dx), C.byref(pc), lam, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh,
            a, vx, vy, T, int(seed), int(stream), int(first), _dev(fresh_sh, torch.complex64) if n_sh > 0 else None,
            _dev(spectrum, torch.complex64), _dev(sh_coef, torch.complex64) if n_sh > 0 else None,
            _dev(screens, torch.float32), _dev(ws), ws.numel()))
        return screens

    # ---- propagation -----------------------------------------------------------------------
    @staticmethod
    def _screen_args(screens, B, N, shared):
        if screens is None:
            return None, 0, 0
        if shared:
            assert screens.dim() == 3
            return screens, 0, screens.shape[0]
        assert screens.dim() == 4 and screens.shape[0] == B
        return screens, screens.shape[1] * N * N, screens.shape[1]

    def propagate(self, N, dx, lam, dz, field, screens=None, shared_screens=False, win_order=0,
                  win_sigma_frac=0.47, n0=1.0, h_kind=H_FRESNEL, out=None, planes=None, stats=None,
                  roi_frac=0.5):
        """field: complex64 [B][N][N]; screens fp32 [B][S][N][N] (or [S][N][N] shared).
        planes: optional complex64 [B][n_steps][N][N]; stats: optional uint8 [B*STATS_BYTES]."""
        B = field.shape[0]
        scr, stride, S = self._screen_args(screens, B, N, shared_screens)
        if out is None:
            out = torch.empty_like(field)
        self._chk(self._lib.ssp_propagate(
            self._h, Grid(N, dx), lam, n0, h_kind, B, len(dz), _host_doubles(dz),
            _dev(scr, torch.float32), stride, S, Window(win_order, win_sigma_frac),
            _dev(field, torch.complex64), _dev(out, torch.complex64), _dev(planes, torch.complex64),
            _dev(stats), roi_frac, None, 0))
        return out

    def evolve_propagate(self, N, dx, psd: PsdParams, lam, cn2, dz, n_sh, a, vx, vy, T, fresh_noise, fresh_noise_sh,
                         spectrum, sh_coef, field, ycol, win_order=16, win_sigma_frac=0.47, n0=1.0, out=None, stats=None,
                         roi_frac=0.5, ws=None):
        """Forward-only temporal frame with the screen synthesis fused into the propagation (N = 1024): advances the AR
        state in place and returns the received fields; ycol: complex64 [B][S][N][N] scratch."""
        B, S = spectrum.shape[0], spectrum.shape[1]
        ws = self.workspace(N, dx, B, S) if ws is None else ws
        if out is None:
            out = torch.empty_like(field)
        pc = psd.c()
        self._chk(self._lib.ssp_evolve_propagate(
            self._h, Grid(N, dx), C.byref(pc), lam, n0, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh, a, vx, vy, T,
            _dev(fresh_noise, torch.complex64), _dev(fresh_noise_sh, torch.complex64) if n_sh > 0 else None,
            _dev(spectrum, torch.complex64), _dev(sh_coef, torch.complex64) if n_sh > 0 else None,
            Window(win_order, win_sigma_frac), _dev(field, torch.complex64), _dev(out, torch.complex64), _dev(stats),
            roi_frac, _dev(ycol, torch.complex64), _dev(ws), ws.numel()))
        return out

    def propagate_adjoint(self, N, dx, lam, dz, g_out, screens=None, shared_screens=False, win_order=0,
                          win_sigma_frac=0.47, n0=1.0, h_kind=H_FRESNEL, out=None, planes=None,
                          phase_grad=None):
        B = g_out.shape[0]
        scr, stride, S = self._screen_args(screens, B, N, shared_screens)
        if out is None:
            out = torch.empty_like(g_out)
        self._chk(self._lib.ssp_propagate_adjoint(
            self._h, Grid(N, dx), lam, n0, h_kind, B, len(dz), _host_doubles(dz),
            _dev(scr, torch.float32), stride, S, Window(win_order, win_sigma_frac),
            _dev(g_out, torch.complex64), _dev(out, torch.complex64), _dev(planes, torch.complex64),
            _dev(phase_grad, torch.float32), None, 0))
        return out

    def beam_stats(self, N, dx, field, roi_frac=0.5, stats=None, mean=None, M2=None, count=None):
        """Returns (stats uint8 tensor [B*STATS_BYTES], new count)."""
        B = field.shape[0]
        if stats is None:
            stats = torch.empty(B * STATS_BYTES, dtype=torch.uint8, device=field.device)
        cnt = C.c_longlong(count if count is not None else 0)
        self._chk(self._lib.ssp_beam_stats(
            self._h, Grid(N, dx), B, _dev(field, torch.complex64), roi_frac, _dev(stats),
            _dev(mean, torch.float32), _dev(M2, torch.float32), C.byref(cnt) if mean is not None else None))
        return stats, cnt.value

    def beam_stats_static(self, N, dx, field, stats, roi_frac=0.5):
        """ssp_beam_stats without allocation (library-resident scratch; B <= STATS_STATIC_MAX_FIELDS): fills the
        caller's stats tensor (uint8 [B*STATS_BYTES], CUDA) and returns it."""
        self._chk(self._lib.ssp_beam_stats_static(
            self._h, Grid(N, dx), field.shape[0], _dev(field, torch.complex64), roi_frac, _dev(stats)))
        return stats

    def propagate_host(self, N, dx, lam, dz, h_field_in, h_field_out, h_screens, shared_screens, S,
                       win_order, win_sigma_frac, h_stats, roi_frac, d_field, d_screens, d_stats,
                       n0=1.0, h_kind=H_FRESNEL):
        """h_*: pinned CPU tensors; d_*: CUDA tensors.  Synchronises the stream."""
        B = d_field.shape[0]
        stride = 0 if (shared_screens or S == 0) else S * N * N
        hp = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        self._chk(self._lib.ssp_propagate_host(
            self._h, Grid(N, dx), lam, n0, h_kind, B, len(dz), _host_doubles(dz),
            hp(h_screens), stride, S, Window(win_order, win_sigma_frac), hp(h_field_in), hp(h_field_out),
            hp(h_stats), roi_frac, _dev(d_field, torch.complex64), _dev(d_screens, torch.float32),
            _dev(d_stats), None, 0))

    def frame_host(self, N, dx, psd: PsdParams, lam, cn2, dz, n_sh, a, vx, vy, T, seed, frame, h_field_in, h_field_out,
                   h_stats, roi_frac, d_field, spectrum, sh_coef, screens, d_noise, d_noise_sh, d_stats, ws,
                   win_order=0, win_sigma_frac=0.0, n0=1.0, h_kind=H_FRESNEL, h_adjoint_out=None, d_adjoint=None):
        """One temporal frame from pinned host fields: device-side noise draws, AR screen evolution, propagation,
        results back on the host.  d_noise: complex64 [frame_chunk(B)][S][N][N] scratch.  h_adjoint_out / d_adjoint:
        also send the received fields back through the screens (A^H U_out) and return that.  Synchronises the stream."""
        B, S = d_field.shape[0], screens.shape[1]
        pc, ar = psd.c(), Ar(a, vx, vy, T, int(seed), int(frame))
        hp = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        self._chk(self._lib.ssp_frame_host(
            self._h, Grid(N, dx), C.byref(pc), lam, n0, h_kind, B, S, _host_doubles(cn2), _host_doubles(dz), n_sh,
            C.byref(ar), Window(win_order, win_sigma_frac), hp(h_field_in), hp(h_field_out), hp(h_stats), roi_frac,
            _dev(d_field, torch.complex64), _dev(spectrum, torch.complex64),
            _dev(sh_coef, torch.complex64) if n_sh > 0 else None, _dev(screens, torch.float32),
            _dev(d_noise, torch.complex64), _dev(d_noise_sh, torch.complex64) if n_sh > 0 else None,
            _dev(d_stats), _dev(ws), ws.numel(), hp(h_adjoint_out), _dev(d_adjoint, torch.complex64)))

    # ---- helpers ---------------------------------------------------------------------------
    def phase_mul(self, N, dx, theta, field, sign=1.0, out=None):
        out = torch.empty_like(field) if out is None else out
        self._chk(self._lib.ssp_phase_mul(self._h, Grid(N, dx), field.shape[0], _dev(theta, torch.float32),
                                          sign, _dev(field, torch.complex64), _dev(out, torch.complex64)))
        return out

    def dft2_centered(self, N, dx, field, inverse=False, out=None):
        out = torch.empty_like(field) if out is None else out
        self._chk(self._lib.ssp_dft2_centered(self._h, Grid(N, dx), field.shape[0], int(inverse),
                                              _dev(field, torch.complex64), _dev(out, torch.complex64), None, 0))
        return out

    def adam_update(self, N, dx, grad, lr, t, m, v, theta, beta1=0.9, beta2=0.999, eps=1e-8):
        """One Adam step (in place on m, v, theta) with the gradient averaged over the batch axis of `grad`."""
        self._chk(self._lib.ssp_adam_update(self._h, Grid(N, dx), grad.shape[0], _dev(grad, torch.float32), float(lr),
                                            float(beta1), float(beta2), float(eps), int(t), _dev(m, torch.float32),
                                            _dev(v, torch.float32), _dev(theta, torch.float32)))

    def fill_noise(self, seed, stream, out, first=0):
        """Fill the complex64 CUDA tensor `out` (any shape, contiguous) with draws first.. of the stream (seed, stream)."""
        self._chk(self._lib.ssp_fill_noise(self._h, int(seed), int(stream), int(first), out.numel(),
                                           _dev(out, torch.complex64)))
        return out

    def philox_words(self, seed, stream, first_block, n_blocks):
        """The generator's raw 32-bit words, int32 CUDA tensor [n_blocks][4] (bit patterns of the unsigned words)."""
        out = torch.empty((int(n_blocks), 4), dtype=torch.int32, device=torch.device("cuda", self.device))
        self._chk(self._lib.ssp_philox_words(self._h, int(seed), int(stream), int(first_block), int(n_blocks),
                                             _dev(out, torch.int32)))
        return out

    def aperture(self, N, dx, radius, field, out=None):
        out = torch.empty_like(field) if out is None else out
        self._chk(self._lib.ssp_aperture(self._h, Grid(N, dx), field.shape[0], float(radius),
                                         _dev(field, torch.complex64), _dev(out, torch.complex64)))
        return out

    def phase_grad(self, N, dx, g, u, out=None):
        out = torch.empty(g.shape, dtype=torch.float32, device=g.device) if out is None else out
        self._chk(self._lib.ssp_phase_grad(self._h, Grid(N, dx), g.shape[0], _dev(g, torch.complex64),
                                           _dev(u, torch.complex64), _dev(out, torch.float32)))
        return out

    def mae_loss(self, N, dx, v, t, grad=None):
        """(loss float64 [B] on the device, gradient complex64 [B][N][N]) of mean |v - t|."""
        B = v.shape[0]
        loss = torch.empty(B, dtype=torch.float64, device=v.device)
        grad = torch.empty_like(v) if grad is None else grad
        self._chk(self._lib.ssp_mae_loss(self._h, Grid(N, dx), B, _dev(v, torch.complex64), _dev(t, torch.complex64),
                                         _dev(loss, torch.float64), _dev(grad, torch.complex64)))
        return loss, grad

    def inner_products(self, N, dx, a, b, out=None):
        out = torch.empty((a.shape[0], 4), dtype=torch.float64, device=a.device) if out is None else out
        self._chk(self._lib.ssp_inner_products(self._h, Grid(N, dx), a.shape[0], _dev(a, torch.complex64),
                                               _dev(b, torch.complex64), _dev(out, torch.float64)))
        return out

    def lincomb(self, N, dx, alpha, a, beta, b, out=None):
        """alpha, beta: python sequences of B complex numbers."""
        B = a.shape[0]
        out = torch.empty_like(a) if out is None else out
        al = _host_doubles([v for z in alpha for v in (complex(z).real, complex(z).imag)])
        be = _host_doubles([v for z in beta for v in (complex(z).real, complex(z).imag)])
        self._chk(self._lib.ssp_lincomb(self._h, Grid(N, dx), B, al, _dev(a, torch.complex64), be,
                                        _dev(b, torch.complex64), _dev(out, torch.complex64)))
        return out


def stats_to_dicts(stats: torch.Tensor):
    """Decode a device uint8 tensor of ssp_stats records (one D2H copy) into python dicts."""
    raw = stats.cpu().numpy().tobytes()
    n = len(raw) // STATS_BYTES
    arr = (Stats * n).from_buffer_copy(raw)
    return [{k: getattr(arr[i], k) for k in STAT_FIELDS} for i in range(n)]
