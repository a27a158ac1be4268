"""GPU: programmatic dependent launch changes nothing but timing.  Every kernel launched with the programmatic-serialization
attribute must wait (griddepcontrol.wait) before it touches another kernel's data; a kernel that did not would read or
overwrite buffers early.  The same frame sequence is run in two fresh processes -- default, and with SSP_NO_PDL=1 (plain
launches) -- and every output must be the same bytes."""
import hashlib
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import hashlib, sys
sys.path.insert(0, %r)
import numpy as np, torch
from paper_2604_07248_b200 import api, d2nn, synth
ctx = api.Context(0)
h = hashlib.sha256()
def add(*ts):
    torch.cuda.synchronize()
    for t in ts:
        h.update(t.detach().cpu().contiguous().numpy().tobytes())
gen = torch.Generator(device="cuda").manual_seed(3)
for N, B, S in ((128, 3, 4), (256, 3, 3), (1024, 3, 3), (2048, 2, 2)):
    dx, lam = 1e-3, 1.0e-6
    dz = [N * dx * dx / lam * 0.2] * S
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    noise = torch.view_as_complex(torch.randn(B, S, N, N, 2, device="cuda", generator=gen))
    nsh = torch.view_as_complex(torch.randn(B, S, 2, 3, 3, 2, device="cuda", generator=gen))
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, 2, 3, 3), dtype=torch.complex64, device="cuda")
    u0 = torch.from_numpy(synth.gaussian_beam(N, dx, 0.1 * N * dx, B)).cuda()
    kw = dict(win_order=16, win_sigma_frac=0.47)
    scr = ctx.make_screens(N, dx, psd, lam, [1e-14] * S, [100.0] * S, 2, noise, nsh, spectrum=spec, sh_coef=shc)
    for frame in range(3):                                   # back to back, no synchronisation inside a frame
        if N >= 512:
            ctx.evolve_screens_seeded(N, dx, psd, lam, [1e-14] * S, [100.0] * S, 2, 0.95, 0.3, -0.2, 1e-2, 9, 2 * frame, 0,
                                      nsh, spec, shc, screens=scr)
        else:
            ctx.evolve_screens(N, dx, psd, lam, [1e-14] * S, [100.0] * S, 2, 0.95, 0.3, -0.2, 1e-2, noise, nsh, spec, shc, screens=scr)
        stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        out = ctx.propagate(N, dx, lam, dz, u0, scr, stats=stats, **kw)
        out_as = ctx.propagate(N, dx, lam, dz, u0, scr, h_kind=api.H_ANGULAR_SPECTRUM, **kw)
        planes = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
        grad = torch.empty((B, S, N, N), dtype=torch.float32, device="cuda")
        out2 = ctx.propagate(N, dx, lam, dz, u0, scr, planes=planes, **kw)
        gin = ctx.propagate_adjoint(N, dx, lam, dz, out2, scr, planes=planes, phase_grad=grad, **kw)
        add(scr, spec, shc, stats, out, out_as, out2, gin, grad)
N, dx, lam, S = 512, 1e-3, 1.55e-6, 4
rx = d2nn.TwoMaskReceiver(ctx, N, dx, lam, [100.0] * S, aperture_radius=0.3 * N * dx, lr=0.01, total_steps=100)
u0 = torch.from_numpy(synth.gaussian_beam(N, dx, 0.1 * N * dx, 2)).cuda()
scr = torch.randn(2, S, N, N, device="cuda", generator=gen) * 0.5
T = rx.target(u0)
for _ in range(5):
    rx.train_step(u0, scr, T=T, sync=False)
add(rx.theta[0], rx.theta[1])
print("HASH", h.hexdigest())
'''


def _run(env_extra):
    env = dict(os.environ)
    env.pop("SSP_NO_PDL", None)
    env.update(env_extra)
    r = subprocess.run([sys.executable, "-c", WORKER % ROOT], capture_output=True, text=True, env=env, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    return [l for l in r.stdout.splitlines() if l.startswith("HASH")][-1]


def test_dependent_launches_change_no_byte():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2604_07248_b200 import build
    build.build()
    assert _run({}) == _run({"SSP_NO_PDL": "1"})
