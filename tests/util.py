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
