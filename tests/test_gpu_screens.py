"""GPU parity: phase-screen generator, AR evolver and the mask-system helpers vs the CPU oracle.

Screen tolerance: relative L2 of one screen <= 2e-5 * log2(N) -- the field
bar of north_star for one screen -- since a screen is one unnormalised inverse 2-D FFT of an
fp32-filtered spectrum plus 8*n_sh fp32 phasor terms."""
import math

import numpy as np
import pytest

from paper_2604_07248_b200 import synth
from tests.util import rel_l2

pytestmark = pytest.mark.gpu

LAM = 1.0e-6


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


def c64(a):
    """float32 [...][2] noise -> complex64 [...] view."""
    return np.ascontiguousarray(a).view(np.complex64)[..., 0]


def _psds(orc):
    from paper_2604_07248_b200 import api
    return {
        "kolmogorov": (orc.Psd(kind=0), api.PsdParams(kind=0)),
        "von_karman": (orc.Psd(kind=1, L0=10.0, l0=5e-3), api.PsdParams(kind=1, L0=10.0, l0=5e-3)),
        "von_karman_592": (orc.Psd(kind=1, L0=3.0, l0=1e-2, km_coeff=5.92),
                           api.PsdParams(kind=1, L0=3.0, l0=1e-2, km_coeff=5.92)),
        "ocean": (orc.Psd(kind=2, chi_T=1e-7, eps=1e-5, w=-2.0), api.PsdParams(kind=2, chi_T=1e-7, eps=1e-5, w=-2.0)),
        # Table S1: biological-tissue exponent, pure power law; and an atmospheric one with both roll-offs
        "power_law": (orc.Psd(kind=3, alpha=4.3, A=2e-16), api.PsdParams(kind=3, alpha=4.3, A=2e-16)),
        "power_law_scales": (orc.Psd(kind=3, alpha=3.5, A=4e-16, L0=5.0, l0=8e-3),
                             api.PsdParams(kind=3, alpha=3.5, A=4e-16, L0=5.0, l0=8e-3)),
    }


@pytest.mark.parametrize("kind", ["kolmogorov", "von_karman", "von_karman_592", "ocean", "power_law", "power_law_scales"])
@pytest.mark.parametrize("N,n_sh", [(32, 3), (128, 3), (256, 0), (512, 2), (1024, 4), (2048, 1)])
def test_make_screens_parity(ssp, orc, kind, N, n_sh):
    import torch
    po, pg = _psds(orc)[kind]
    ocean = kind == "ocean"
    dx, lam = (2.5e-4, 0.532e-6) if ocean else (2e-3, LAM)
    B, S = (2, 3) if N <= 256 else (1, 2)
    cn2 = [1e-14, 3e-14, 2e-15][:S]
    dz = [100.0, 40.0, 250.0][:S] if not ocean else [2.5, 1.0, 4.0][:S]
    hi, sh = synth.noise_batch(40 + N, 0, B, S, N, n_sh)
    ref, spec_ref, shc_ref = orc.make_screens(N, dx, po, lam, cn2, dz, n_sh, hi, sh if n_sh else None)
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device="cuda")
    scr = ssp.make_screens(N, dx, pg, lam, cn2, dz, n_sh, cu(c64(hi)), cu(c64(sh)) if n_sh else None,
                           spectrum=spec, sh_coef=shc if n_sh else None)
    err = rel_l2(scr.cpu().numpy(), ref)
    assert err.max() < 2e-5 * math.log2(N), err
    assert rel_l2(spec.cpu().numpy(), spec_ref).max() < 5e-6
    if n_sh:
        assert np.abs(shc.cpu().numpy() - shc_ref).max() < 1e-6 * np.abs(shc_ref).max()
    # outputs that may be NULL really are optional, and give the same screens
    scr2 = ssp.make_screens(N, dx, pg, lam, cn2, dz, n_sh, cu(c64(hi)), cu(c64(sh)) if n_sh else None)
    assert torch.equal(scr, scr2)
    assert abs(float(scr.mean())) < 1e-4 * float(scr.abs().max())    # piston removed


def test_screen_statistics_on_gpu(ssp, orc):
    """Property at a size the oracle cannot sweep: variance of GPU screens = sum_k s_k^2 (S16 normalisation)."""
    from paper_2604_07248_b200 import api
    N, dx, B, S = 512, 4e-3, 4, 8
    po = orc.Psd(kind=1, L0=2.0, l0=1e-2)
    pg = api.PsdParams(kind=1, L0=2.0, l0=1e-2)
    hi, _ = synth.noise_batch(77, 0, B, S, N, 0)
    scr = ssp.make_screens(N, dx, pg, LAM, [1e-14] * S, [100.0] * S, 0, cu(c64(hi)))
    k = np.arange(N)
    f = np.where(k < N // 2, k, k - N) / (N * dx)
    fx, fy = np.meshgrid(f, f)
    df = 1.0 / (N * dx)
    expect = np.sum(orc.psd_f(po, LAM, 1e-14, 100.0, np.hypot(fx, fy))) * df * df
    var = float(scr.double().var())
    assert abs(var / expect - 1) < 0.05, (var, expect)


def test_evolve_screens_parity(ssp, orc):
    import torch
    from paper_2604_07248_b200 import api
    N, dx, n_sh, B, S = 64, 2e-3, 3, 2, 2
    po, pg = orc.Psd(kind=1, L0=10.0, l0=5e-3), api.PsdParams(kind=1, L0=10.0, l0=5e-3)
    cn2, dz = [1e-14, 2e-14], [100.0, 60.0]
    hi0, sh0 = synth.noise_batch(50, 0, B, S, N, n_sh, frame=0)
    _, spec_ref, shc_ref = orc.make_screens(N, dx, po, LAM, cn2, dz, n_sh, hi0, sh0)
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, n_sh, 3, 3), dtype=torch.complex64, device="cuda")
    ssp.make_screens(N, dx, pg, LAM, cn2, dz, n_sh, cu(c64(hi0)), cu(c64(sh0)), spectrum=spec, sh_coef=shc)
    a, T = 0.99, 0.01
    vx, vy = 3 * dx / T * 0.37, -1.3 * dx / T                  # fractional-pixel wind
    for frame in (1, 2, 3):
        hin, shn = synth.noise_batch(50, 0, B, S, N, n_sh, frame=frame)
        ref = orc.evolve_screens(N, dx, po, LAM, cn2, dz, n_sh, a, vx, vy, T, hin, shn, spec_ref, shc_ref)
        scr = ssp.evolve_screens(N, dx, pg, LAM, cn2, dz, n_sh, a, vx, vy, T, cu(c64(hin)), cu(c64(shn)), spec, shc)
        err = rel_l2(scr.cpu().numpy(), ref)
        assert err.max() < 2e-5 * math.log2(N) * (frame + 1), (frame, err)
    # a = 1, v = 0 leaves the screen unchanged; a = 0 gives the fresh screen
    before = ssp.evolve_screens(N, dx, pg, LAM, cn2, dz, n_sh, 1.0, 0, 0, 0, cu(c64(hin)), cu(c64(shn)), spec, shc)
    assert rel_l2(before.cpu().numpy(), scr.cpu().numpy()).max() < 1e-6
    fresh = ssp.make_screens(N, dx, pg, LAM, cn2, dz, n_sh, cu(c64(hin)), cu(c64(shn)))
    after = ssp.evolve_screens(N, dx, pg, LAM, cn2, dz, n_sh, 0.0, 0, 0, 0, cu(c64(hin)), cu(c64(shn)), spec, shc)
    assert rel_l2(after.cpu().numpy(), fresh.cpu().numpy()).max() < 1e-6
    with pytest.raises(api.SspError) as e:
        ssp.evolve_screens(N, dx, pg, LAM, cn2, dz, n_sh, 1.5, 0, 0, 0, cu(c64(hin)), cu(c64(shn)), spec, shc)
    assert e.value.code == api.EINVAL
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(api.SspError) as e:
        ssp.make_screens(N, dx, pg, LAM, cn2, dz, n_sh, cu(c64(hin)), cu(c64(shn)), ws=small)
    assert e.value.code == api.EWORKSPACE


@pytest.mark.parametrize("N,n_sh,kind", [(512, 3, 1), (4096, 3, 1), (512, 2, 2)])
def test_evolve_screens_wind_and_subharmonics_large_grids(ssp, orc, N, n_sh, kind):
    """AR evolution with wind AND subharmonics against the oracle on the grids whose kernels round 1 never compared
    under AR: 512 (k_screen_col_tma<512,.,AR,TILT>) and 4096 (register-load generator, (32,16,8) plan); fractional-pixel
    wind with vx != vy; von Karman and (512) the oceanic filter.  One stack of one screen, two AR frames at 512, one at
    4096 (the oracle needs about half a minute per 4096^2 screen)."""
    import torch
    from paper_2604_07248_b200 import api
    from tests.util import record
    dx, B, S = 1e-3, 1, 1
    if kind == 1:
        po, pg = orc.Psd(kind=1, L0=20.0, l0=4e-3), api.PsdParams(kind=1, L0=20.0, l0=4e-3)
    else:
        po = orc.Psd(kind=2, chi_T=1e-7, eps=1e-5, w=-2.0)
        pg = api.PsdParams(kind=2, chi_T=1e-7, eps=1e-5, w=-2.0)
    cn2, dz = [3e-14], [120.0]
    frames = synth.noise(80 + N, kind, 0, S, N, n_sh, frames=3 if N <= 512 else 2)
    hi0, sh0 = frames[0]
    _, spec_ref, shc_ref = orc.make_screens(N, dx, po, LAM, cn2, dz, n_sh, hi0[None], sh0[None])
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, n_sh, 3, 3), dtype=torch.complex64, device="cuda")
    ssp.make_screens(N, dx, pg, LAM, cn2, dz, n_sh, cu(c64(hi0[None])), cu(c64(sh0[None])), spectrum=spec, sh_coef=shc)
    a, T = 0.95, 0.02
    vx, vy = 2.37 * dx / T, -0.61 * dx / T
    for t in range(1, len(frames)):
        hi, sh = frames[t]
        ref = orc.evolve_screens(N, dx, po, LAM, cn2, dz, n_sh, a, vx, vy, T, hi[None], sh[None], spec_ref, shc_ref)
        scr = ssp.evolve_screens(N, dx, pg, LAM, cn2, dz, n_sh, a, vx, vy, T, cu(c64(hi[None])), cu(c64(sh[None])), spec, shc)
        err = rel_l2(scr.cpu().numpy(), ref).max()
        record("evolve_wind_sh", N=N, kind=kind, frame=t, screens=float(err), bound=2e-5 * math.log2(N) * (t + 1))
        assert err < 2e-5 * math.log2(N) * (t + 1), (t, err)
        # the stored AR state too: spectrum and subharmonic coefficients
        es = np.linalg.norm(spec.cpu().numpy() - spec_ref) / np.linalg.norm(spec_ref)
        ec = np.linalg.norm(shc.cpu().numpy() - shc_ref) / np.linalg.norm(shc_ref)
        assert es < 1e-6 * (t + 1) and ec < 1e-6 * (t + 1), (es, ec)


def test_ar_chain_100_steps(ssp, orc):
    """Config-3 style AR chain on one screen: 100 steps at a = 0.99, GPU fp32 state vs oracle fp64 state."""
    import torch
    from paper_2604_07248_b200 import api
    N, dx, n_sh = 64, 1e-3, 3
    po, pg = orc.Psd(kind=1, L0=20.0, l0=2e-3), api.PsdParams(kind=1, L0=20.0, l0=2e-3)
    cn2, dz = [5e-15], [150.0]
    frames = synth.noise(3, 0, 0, 1, N, n_sh, frames=101)
    hi0, sh0 = frames[0]
    _, spec_ref, shc_ref = orc.make_screens(N, dx, po, 1.55e-6, cn2, dz, n_sh, hi0[None], sh0[None])
    spec = torch.empty((1, 1, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((1, 1, n_sh, 3, 3), dtype=torch.complex64, device="cuda")
    ssp.make_screens(N, dx, pg, 1.55e-6, cn2, dz, n_sh, cu(c64(hi0[None])), cu(c64(sh0[None])), spectrum=spec, sh_coef=shc)
    for t in range(1, 101):
        hi, sh = frames[t]
        ref = orc.evolve_screens(N, dx, po, 1.55e-6, cn2, dz, n_sh, 0.99, 0, 0, 0, hi[None], sh[None], spec_ref, shc_ref)
        scr = ssp.evolve_screens(N, dx, pg, 1.55e-6, cn2, dz, n_sh, 0.99, 0, 0, 0, cu(c64(hi[None])), cu(c64(sh[None])), spec, shc)
    # the recursion is a contraction (a < 1): rounding does not accumulate
    assert rel_l2(scr.cpu().numpy(), ref).max() < 2e-5 * math.log2(N) * 2


def test_mask_system_helpers(ssp, orc):
    N, dx, B = 64, 1e-3, 2
    u = synth.random_field(N, B, 61)
    v = synth.random_field(N, B, 62)
    th = synth.phase_masks(0, N, 1)[0]
    for N2 in (8, 64, 256, 512, 1024, 4096):
        w = synth.random_field(N2, B, 63)
        F = ssp.dft2_centered(N2, dx, cu(w))
        assert rel_l2(F.cpu().numpy(), orc.dft2_centered(N2, w)).max() < 2e-5 * math.log2(N2)
        back = ssp.dft2_centered(N2, dx, F, inverse=True)
        assert rel_l2(back.cpu().numpy(), w.astype(np.complex128)).max() < 2e-5 * math.log2(N2)
    pm = ssp.phase_mul(N, dx, cu(th), cu(u))
    assert rel_l2(pm.cpu().numpy(), orc.phase_mul(N, th, u)).max() < 2e-6
    pm = ssp.phase_mul(N, dx, cu(th), cu(u), sign=-1.0)
    assert rel_l2(pm.cpu().numpy(), orc.phase_mul(N, th, u, sign=-1.0)).max() < 2e-6
    g = ssp.phase_grad(N, dx, cu(u), cu(v)).cpu().numpy()
    np.testing.assert_allclose(g, orc.phase_grad(N, u, v), rtol=0, atol=2e-6 * np.abs(u).max() * np.abs(v).max())
    ip = ssp.inner_products(N, dx, cu(u), cu(v)).cpu().numpy()
    for b in range(B):
        ref = np.vdot(u[b].astype(np.complex128), v[b].astype(np.complex128))
        assert abs(complex(ip[b, 0], ip[b, 1]) - ref) < 1e-9 * N * N
        assert abs(ip[b, 2] - np.sum(np.abs(u[b].astype(np.complex128)) ** 2)) < 1e-9 * N * N
        assert abs(ip[b, 3] - np.sum(np.abs(v[b].astype(np.complex128)) ** 2)) < 1e-9 * N * N
    al, be = [0.5 - 2j, 1.25 + 0.5j], [-1 + 0.25j, 3.0]
    lc = ssp.lincomb(N, dx, al, cu(u), be, cu(v)).cpu().numpy()
    ref = np.stack([al[b] * u[b].astype(np.complex128) + be[b] * v[b].astype(np.complex128) for b in range(B)])
    assert rel_l2(lc, ref).max() < 1e-6


@pytest.mark.parametrize("N,n_sh", [(64, 3), (1024, 3), (2048, 0)])
def test_paired_screens_parity(ssp, orc, N, n_sh):
    """ssp_make_screens_pair / ssp_evolve_screens_pair: the imaginary part of each synthesis as a second screen
    (oracle: orc.synthesize(part="im"), pinned to the real-part path on the CPU)."""
    import torch
    from paper_2604_07248_b200 import api
    dx, B, S = 2e-3, 1, 2
    po, pg = orc.Psd(kind=1, L0=10.0, l0=5e-3), api.PsdParams(kind=1, L0=10.0, l0=5e-3)
    cn2, dz = [1e-14, 3e-14], [100.0, 40.0]
    hi, sh = synth.noise_batch(60 + N, 0, B, S, N, n_sh)
    ref, spec_ref, shc_ref = orc.make_screens(N, dx, po, LAM, cn2, dz, n_sh, hi, sh if n_sh else None)
    ref_im = orc.synthesize(N, dx, n_sh, spec_ref, shc_ref, part="im")
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device="cuda")
    im = torch.empty((B, S, N, N), dtype=torch.float32, device="cuda")
    scr = ssp.make_screens(N, dx, pg, LAM, cn2, dz, n_sh, cu(c64(hi)), cu(c64(sh)) if n_sh else None,
                           spectrum=spec, sh_coef=shc if n_sh else None, screens_im=im)
    bound = 2e-5 * math.log2(N)
    assert rel_l2(scr.cpu().numpy(), ref).max() < bound
    assert rel_l2(im.cpu().numpy(), ref_im).max() < bound
    # one AR step with wind: both screens follow the stored spectrum
    hin, shn = synth.noise_batch(60 + N, 0, B, S, N, n_sh, frame=1)
    a, T = 0.97, 0.01
    vx, vy = 2.3 * dx / T, -0.7 * dx / T
    ref2 = orc.evolve_screens(N, dx, po, LAM, cn2, dz, n_sh, a, vx, vy, T, hin, shn if n_sh else None, spec_ref, shc_ref)
    ref2_im = orc.synthesize(N, dx, n_sh, spec_ref, shc_ref, part="im")      # spec_ref / shc_ref were advanced in place
    scr2 = ssp.evolve_screens(N, dx, pg, LAM, cn2, dz, n_sh, a, vx, vy, T, cu(c64(hin)), cu(c64(shn)) if n_sh else None,
                              spec, shc if n_sh else None, screens_im=im)
    assert rel_l2(scr2.cpu().numpy(), ref2).max() < 2 * bound
    assert rel_l2(im.cpu().numpy(), ref2_im).max() < 2 * bound
