"""GPU parity of the two-mask receiver (paper_2604_07248_b200/d2nn.py) against the CPU oracle
chain of tests/o9.py, of the Adam update against orc.adam_step, and a short training run on fresh turbulence."""
import math

import numpy as np
import pytest

from paper_2604_07248_b200 import synth
from tests import o9
from tests.util import rel_l2

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ssp():
    import torch
    from paper_2604_07248_b200 import api, build
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    ctx = api.Context(0)
    yield ctx
    ctx.close()


def cu(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("loss_kind", ["mae", "overlap"])
@pytest.mark.parametrize("N,R", [(64, None), (64, 1.9e-2), (256, 8.3e-2)])
def test_receiver_loss_and_gradients(ssp, orc, N, R, loss_kind):
    """Both losses: the paper's mean absolute error (ssp_mae_loss) and config 4's overlap loss."""
    from paper_2604_07248_b200 import d2nn
    dx, lam, B, S = 1e-3, 1e-6, 2, 3
    rng = np.random.default_rng(N)
    dz = (N * dx * dx / lam) * (0.05 + 0.1 * rng.random(S))
    u0 = synth.gaussian_beam(N, dx, 0.12 * N * dx, B)
    scr = synth.random_screens(N, B, S, 5 + N, rms=1.5)
    th = synth.phase_masks(1, N, 2)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    ref = o9.oracle_chain(orc, N, dx, lam, dz, u0, scr, th[0], th[1], kw, aperture_radius=R, loss_kind=loss_kind)
    rx = d2nn.TwoMaskReceiver(ssp, N, dx, lam, list(dz), aperture_radius=R, theta=[cu(th[0]), cu(th[1])], loss=loss_kind)
    loss, g1, g2, G0 = rx.loss_and_grads(cu(u0), cu(scr), input_grad=True)
    np.testing.assert_allclose(loss, ref["loss"], rtol=2e-4, atol=1e-6)
    bound = 2e-5 * math.log2(N) * (2 * S + 4)
    assert rel_l2(g1.cpu().numpy(), ref["g_th1"]).max() < bound
    assert rel_l2(g2.cpu().numpy(), ref["g_th2"]).max() < bound
    assert rel_l2(G0.cpu().numpy(), ref["G0"]).max() < bound


def test_adam_update_parity(ssp, orc):
    import torch
    N, B = 64, 3
    rng = np.random.default_rng(9)
    th = rng.standard_normal((N, N)).astype(np.float32)
    m = np.zeros((N, N)); v = np.zeros((N, N)); th_ref = th.astype(np.float64)
    d_m, d_v, d_th = cu(m.astype(np.float32)), cu(v.astype(np.float32)), cu(th)
    for t in range(1, 6):
        g = (rng.standard_normal((B, N, N)) * 10.0 ** rng.uniform(-4, 0)).astype(np.float32)
        m, v, th_ref = orc.adam_step(g, 0.01, t, m, v, th_ref)
        ssp.adam_update(N, 1e-3, cu(g), 0.01, t, d_m, d_v, d_th)
        np.testing.assert_allclose(d_th.cpu().numpy(), th_ref, rtol=0, atol=2e-6)
        # fp32 state against the fp64 recursion: a few ulp of the largest term (m is a signed sum: cancellation)
        np.testing.assert_allclose(d_m.cpu().numpy(), m, rtol=1e-5, atol=1e-6 * np.abs(m).max())
        np.testing.assert_allclose(d_v.cpu().numpy(), v, rtol=1e-5, atol=1e-6 * np.abs(v).max())


@pytest.mark.parametrize("loss_kind,floor", [("mae", 0.0), ("overlap", 0.2)])
def test_training_reduces_the_loss_on_fresh_turbulence(ssp, loss_kind, floor):
    """Sec. 2.5 in miniature: every epoch draws new screens (make_screens on device noise).  The transmitted beam
    carries a static defocus that the target (the clean beam propagated in vacuum) does not: the two masks learn to
    undo it through weak turbulence, so the mean loss falls well below that of the untrained receiver -- with the
    paper's mean-absolute-error loss (the default) and with the overlap loss."""
    import torch
    from paper_2604_07248_b200 import api, d2nn
    N, dx, lam, S, B = 128, 1e-3, 1.064e-6, 3, 8
    dz = [300.0] * S
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    clean = synth.gaussian_beam(N, dx, 1.5e-2, B)
    x = synth.coords(N, dx)
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    u0 = cu((clean * np.exp(1j * 2.5 * r2 / (1.5e-2) ** 2)).astype(np.complex64))
    rx = d2nn.TwoMaskReceiver(ssp, N, dx, lam, dz, aperture_radius=5e-2, lr=0.02, total_steps=150, loss=loss_kind)
    T = rx.target(cu(clean))
    gen = torch.Generator(device="cuda")

    def fresh():
        noise = torch.view_as_complex(torch.randn(B, S, N, N, 2, device="cuda", generator=gen))
        nsh = torch.view_as_complex(torch.randn(B, S, 3, 3, 3, 2, device="cuda", generator=gen))
        return ssp.make_screens(N, dx, psd, lam, [2e-15] * S, dz, 3, noise, nsh)

    gen.manual_seed(3)
    base = np.mean([rx.loss_and_grads(u0, fresh(), T)[0].mean() for _ in range(10)])
    losses = [rx.train_step(u0, fresh(), T) for _ in range(150)]
    gen.manual_seed(3)                                          # the same ten draws as `base`
    after = np.mean([rx.loss_and_grads(u0, fresh(), T)[0].mean() for _ in range(10)])
    assert base > floor, base                                   # the defocus does spoil the received field
    assert after < (0.5 if loss_kind == "overlap" else 0.7) * base, (base, after, losses[-5:])
