"""Shared test helpers (no method arithmetic)."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def paper_constants():
    out = {}
    with open(os.path.join(GOLDEN, "paper_constants.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()
                out[k] = float(v)
    return out


def rel_l2(a, b):
    """Per-field relative L2 error of a against reference b (fields on the last two axes)."""
    a = np.asarray(a)
    b = np.asarray(b)
    num = np.sqrt(np.sum(np.abs(a.astype(np.complex128) - b) ** 2, axis=(-2, -1)))
    den = np.sqrt(np.sum(np.abs(b) ** 2, axis=(-2, -1)))
    return num / np.maximum(den, 1e-300)


def pmap(fn, items, workers=None):
    """Run independent oracle calls side by side (threads: ctypes releases the GIL inside the C oracle, and every
    oracle call works on buffers of its own).  The oracle itself is untouched -- this only issues several of its
    calls at once so that the full-size parity tests finish within the GPU-test budget."""
    from concurrent.futures import ThreadPoolExecutor
    items = list(items)
    n = min(len(items), workers or (os.cpu_count() or 1))
    if n <= 1:
        return [fn(x) for x in items]
    with ThreadPoolExecutor(max_workers=n) as ex:
        return list(ex.map(fn, items))


def oracle_screens_parallel(orc, N, dx, psd, lam, cn2, dz, n_sh, hi, sh, keep_spectrum=False):
    """orc.make_screens called once per (b, s) screen, side by side; same results as one call on the whole array."""
    B, S = hi.shape[0], hi.shape[1]

    def one(bs):
        b, s = divmod(bs, S)
        return orc.make_screens(N, dx, psd, lam, [cn2[s]], [dz[s]], n_sh, hi[b:b + 1, s:s + 1],
                                sh[b:b + 1, s:s + 1] if n_sh > 0 else None, keep_spectrum=keep_spectrum)
    res = pmap(one, range(B * S))
    scr = np.stack([r[0][0, 0] for r in res]).reshape(B, S, N, N)
    spec = np.stack([r[1][0, 0] for r in res]).reshape(B, S, N, N) if keep_spectrum else None
    shc = np.stack([r[2][0, 0] for r in res]).reshape(B, S, -1, 3, 3) if n_sh > 0 else None
    return scr, spec, shc


def record(name, **vals):
    """Append measured parity errors to gpurun_out/parity_errors.txt when that folder exists (the numbers DESIGN.md quotes)."""
    d = os.path.join(os.path.dirname(GOLDEN.rstrip("/")), "..", "gpurun_out")
    d = os.path.normpath(d)
    if os.path.isdir(d):
        try:
            with open(os.path.join(d, "parity_errors.txt"), "a") as fh:
                fh.write(name + " " + " ".join(f"{k}={v:.3e}" if isinstance(v, float) else f"{k}={v}" for k, v in vals.items()) + "\n")
        except OSError:
            pass
