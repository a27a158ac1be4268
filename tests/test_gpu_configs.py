"""GPU parity on BASELINE.json configs 2-5 at the slices SURVEY.md 8(d) states (config 1 runs in full in
test_gpu_propagate.py) and on the bench launch configuration at full size.

Slices: the grid, geometry, medium, beam, batch layout AND the number of screens / split steps are the config's own;
what is cut is the number of realisations (config 2: 4 of 64 per Cn2; config 3: 2 of 32 stacks and 3 of 100 AR frames;
configs 4 and 5: B = 1) -- the fp64 oracle needs 2.8 s / 12 s per split step at 2048^2 / 4096^2.  Independent oracle
calls (one per screen, forward / vacuum legs) are issued side by side from threads (tests/util.py: pmap).
Bar: per-field relative L2 <= 2e-5 log2(N) screens (north_star); screens 2e-5 log2(N) each."""
import math

import numpy as np
import pytest

from paper_2604_07248_b200 import synth
from tests.util import oracle_screens_parallel, pmap, record, rel_l2

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


def c64(a):
    return np.ascontiguousarray(a).view(np.complex64)[..., 0]


def tol(N, n):
    return 2e-5 * math.log2(N) * max(1, n)


def _psd(wl, orc):
    from paper_2604_07248_b200 import api
    return orc.Psd(**wl.psd_dict()), api.PsdParams(**wl.psd_dict())


def _check_stats(st, st_ref, wl):
    for a, b in zip(st, st_ref):
        for k in ("power", "w2", "sxx", "syy", "roi_sumI", "roi_sumI2", "I_axis"):
            assert abs(a[k] / b[k] - 1) < 1e-4, (k, a[k], b[k])
        assert abs(a["cx"] - b["cx"]) < 1e-4 * wl.dx * wl.N and abs(a["cy"] - b["cy"]) < 1e-4 * wl.dx * wl.N
        assert a["roi_n"] == b["roi_n"]


def test_config2_scintillation_sweep_slice(ssp, orc):
    """configs[1]: 512^2 plane wave, 10 Kolmogorov screens, Cn2 in {1e-15, 1e-14, 1e-13}; slice = 4 of the 64
    realisations per Cn2.  Screens, received field and the ROI sums behind the scintillation index."""
    import torch
    from paper_2604_07248_b200 import api
    wl = synth.CONFIGS[2]
    N, S, B = wl.N, wl.S, 4
    po, pg = _psd(wl, orc)
    u0 = synth.input_field(wl, B)
    for ic, cn2 in enumerate(wl.cn2_sweep):
        hi, sh = synth.noise_batch(2, ic, B, S, N, 0)
        cn2s = np.full(S, cn2)
        scr_ref, _, _ = oracle_screens_parallel(orc, N, wl.dx, po, wl.lam, cn2s, wl.dz, 0, hi, sh)
        scr = ssp.make_screens(N, wl.dx, pg, wl.lam, list(cn2s), list(wl.dz), 0, cu(c64(hi)))
        e_scr = rel_l2(scr.cpu().numpy(), scr_ref).max()
        assert e_scr < tol(N, 1)
        scr32 = scr_ref.astype(np.float32)                    # identical fp32 screens feed both propagators
        kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
        ref = np.concatenate(pmap(lambda b: orc.propagate(N, wl.dx, wl.lam, wl.dz, u0[b:b + 1], scr32[b:b + 1], **kw), range(B)))
        stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        out = ssp.propagate(N, wl.dx, wl.lam, list(wl.dz), cu(u0), cu(scr32), stats=stats, roi_frac=0.5, **kw)
        err = rel_l2(out.cpu().numpy(), ref)
        assert err.max() < tol(N, S), (cn2, err)
        record("config2", cn2=float(cn2), B=B, S=S, screens=float(e_scr), field=float(err.max()), bound=tol(N, S))
        _check_stats(api.stats_to_dicts(stats), orc.beam_stats(N, wl.dx, ref, roi_frac=0.5), wl)


def test_config3_temporal_slice(ssp, orc):
    """configs[2]: 1024^2, 20 von Karman screens + 3 subharmonic levels, AR a = 0.99, Gaussian beam; slice = 2 of
    the 32 stacks x 3 of the 100 AR frames.  Per frame: every evolved screen, the received fields, the
    beam statistics.  (The 100-step AR chain on one screen is test_gpu_screens.py::test_ar_chain_100_steps.)"""
    import torch
    from paper_2604_07248_b200 import api
    wl = synth.CONFIGS[3]
    N, S, B, T = wl.N, wl.S, 2, 3
    po, pg = _psd(wl, orc)
    frames = [synth.noise(3, 0, b, S, N, wl.n_sh, frames=T + 1) for b in range(B)]          # [b][t] -> (hi, sh)
    hi = lambda t: np.stack([frames[b][t][0] for b in range(B)])
    sh = lambda t: np.stack([frames[b][t][1] for b in range(B)])
    _, spec_ref, shc_ref = oracle_screens_parallel(orc, N, wl.dx, po, wl.lam, wl.cn2_list, wl.dz, wl.n_sh, hi(0), sh(0),
                                                   keep_spectrum=True)
    spec_ref, shc_ref = np.ascontiguousarray(spec_ref), np.ascontiguousarray(shc_ref)
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, wl.n_sh, 3, 3), dtype=torch.complex64, device="cuda")
    ssp.make_screens(N, wl.dx, pg, wl.lam, list(wl.cn2_list), list(wl.dz), wl.n_sh, cu(c64(hi(0))), cu(c64(sh(0))),
                     spectrum=spec, sh_coef=shc)
    u0 = synth.input_field(wl, B)
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    for t in range(1, T + 1):
        h_t, s_t = hi(t), sh(t)

        def evolve_one(bs):                                    # one (stack, screen) at a time: the AR state is per screen
            b, j = divmod(bs, S)
            sp, sc = np.ascontiguousarray(spec_ref[b:b + 1, j:j + 1]), np.ascontiguousarray(shc_ref[b:b + 1, j:j + 1])
            out = orc.evolve_screens(N, wl.dx, po, wl.lam, [wl.cn2_list[j]], [wl.dz[j]], wl.n_sh, wl.ar_a, 0, 0, 0,
                                     h_t[b:b + 1, j:j + 1], s_t[b:b + 1, j:j + 1], sp, sc)
            return out[0, 0], sp[0, 0], sc[0, 0]
        res = pmap(evolve_one, range(B * S))
        scr_ref = np.stack([r[0] for r in res]).reshape(B, S, N, N)
        spec_ref = np.stack([r[1] for r in res]).reshape(B, S, N, N)
        shc_ref = np.stack([r[2] for r in res]).reshape(B, S, wl.n_sh, 3, 3)
        scr = ssp.evolve_screens(N, wl.dx, pg, wl.lam, list(wl.cn2_list), list(wl.dz), wl.n_sh, wl.ar_a, 0, 0, 0,
                                 cu(c64(h_t)), cu(c64(s_t)), spec, shc)
        e_scr = rel_l2(scr.cpu().numpy(), scr_ref)
        assert e_scr.max() < tol(N, t + 1), (t, e_scr)
        scr32 = scr_ref.astype(np.float32)
        ref = np.concatenate(pmap(lambda b: orc.propagate(N, wl.dx, wl.lam, wl.dz, u0[b:b + 1], scr32[b:b + 1], **kw), range(B)))
        stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        out = ssp.propagate(N, wl.dx, wl.lam, list(wl.dz), cu(u0), cu(scr32), stats=stats, roi_frac=0.25, **kw)
        e_f = rel_l2(out.cpu().numpy(), ref)
        assert e_f.max() < tol(N, S), (t, e_f)
        record("config3", frame=t, B=B, S=S, screens=float(e_scr.max()), field=float(e_f.max()), bound=tol(N, S))
        _check_stats(api.stats_to_dicts(stats), orc.beam_stats(N, wl.dx, ref, roi_frac=0.25), wl)


def test_config4_forward_adjoint_masks_all_screens(ssp, orc):
    """configs[3] at its own step count: 2048^2, all 30 Kolmogorov Cn2 = 1e-13 screens at dz = L/30, Gaussian beam, two
    uniform-random phase masks (receiver pupil, Fourier plane of a 2f system), Gaussian-overlap loss and its gradients
    w.r.t. both masks and every one of the 30 screens via the adjoint split step.  Slice = 1 of the 8 fields."""
    from tests import o9
    wl = synth.CONFIGS[4]
    N, S, B = wl.N, wl.S, 1
    po, pg = _psd(wl, orc)
    dz, cn2 = wl.dz, wl.cn2_list
    hi, sh = synth.noise_batch(4, 0, B, S, N, 0)
    scr_ref, _, _ = oracle_screens_parallel(orc, N, wl.dx, po, wl.lam, cn2, dz, 0, hi, sh)
    scr = ssp.make_screens(N, wl.dx, pg, wl.lam, list(cn2), list(dz), 0, cu(c64(hi)))
    e_scr = rel_l2(scr.cpu().numpy(), scr_ref).max()
    assert e_scr < tol(N, 1)
    del hi, scr
    scr32 = scr_ref.astype(np.float32)
    del scr_ref
    th = synth.phase_masks(0, N, 2)
    u0 = synth.input_field(wl, B)
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    ref = o9.oracle_chain(orc, N, wl.dx, wl.lam, dz, u0, scr32, th[0], th[1], kw, parallel=True)
    got = o9.gpu_chain(ssp, N, wl.dx, wl.lam, dz, u0, scr32, th[0], th[1], kw)
    e = dict(V5=rel_l2(got["V5"].cpu().numpy(), ref["V5"]).max(), G0=rel_l2(got["G0"].cpu().numpy(), ref["G0"]).max(),
             g_th1=rel_l2(got["g_th1"].cpu().numpy(), ref["g_th1"]).max(),
             g_th2=rel_l2(got["g_th2"].cpu().numpy(), ref["g_th2"]).max(),
             g_phi=rel_l2(got["g_phi"].cpu().numpy(), ref["g_phi"]).max())
    record("config4", B=B, S=S, screens=float(e_scr), loss_gpu=float(got["loss"][0]), loss_ref=float(ref["loss"][0]),
           bound_fwd=tol(N, S + 2), bound_bwd=tol(N, 2 * S + 4), **{k: float(v) for k, v in e.items()})
    assert e["V5"] < tol(N, S + 2), e
    assert abs(got["loss"][0] - ref["loss"][0]) < 1e-4 * max(ref["loss"][0], 1e-3), (got["loss"], ref["loss"])
    for k in ("G0", "g_th1", "g_th2", "g_phi"):
        assert e[k] < tol(N, 2 * S + 4), (k, e)


def test_config5_ocean_all_screens(ssp, orc):
    """configs[4] at its own step count: 4096^2, all 20 Nikishov oceanic screens with 4 subharmonic levels, Gaussian
    beam w0 = 5 mm, dz = L/20.  Slice = 1 of the 2 fields.  Every screen, the received field, the beam statistics."""
    import torch
    from paper_2604_07248_b200 import api
    wl = synth.CONFIGS[5]
    N, S, B = wl.N, wl.S, 1
    po, pg = _psd(wl, orc)
    dz, cn2 = wl.dz, wl.cn2_list
    hi, sh = synth.noise_batch(5, 0, B, S, N, wl.n_sh)
    scr = ssp.make_screens(N, wl.dx, pg, wl.lam, list(cn2), list(dz), wl.n_sh, cu(c64(hi)), cu(c64(sh))).cpu().numpy()
    scr_ref, _, _ = oracle_screens_parallel(orc, N, wl.dx, po, wl.lam, cn2, dz, wl.n_sh, hi, sh)
    e_scr = rel_l2(scr, scr_ref)
    assert e_scr.max() < tol(N, 1), e_scr
    del hi, scr
    scr32 = scr_ref.astype(np.float32)
    del scr_ref
    u0 = synth.input_field(wl, B)
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    out = ssp.propagate(N, wl.dx, wl.lam, list(dz), cu(u0), cu(scr32), stats=stats, roi_frac=0.25, **kw).cpu().numpy()
    ref = orc.propagate(N, wl.dx, wl.lam, dz, u0, scr32, **kw)
    e_f = rel_l2(out, ref).max()
    record("config5", B=B, S=S, screens=float(e_scr.max()), field=float(e_f), bound=tol(N, S))
    assert e_f < tol(N, S)
    _check_stats(api.stats_to_dicts(stats), orc.beam_stats(N, wl.dx, ref, roi_frac=0.25), wl)


def test_bench_launch_configuration_full_size(ssp, orc):
    """The launch configuration bench.py times (config 3 in full: 1024^2, B = 32 stacks of 20 screens, one AR
    frame with the seeded generator): realisation 17 of the batch is checked against the oracle run on that realisation alone (screens,
    received field, adjoint field); properties that hold at any size cover the rest of the batch."""
    import torch
    from paper_2604_07248_b200 import api
    wl = synth.CONFIGS[3]
    N, S, B, b_s = wl.N, wl.S, wl.B, 17
    po, pg = _psd(wl, orc)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(7)
    noise = [torch.view_as_complex(torch.randn(B, S, N, N, 2, device="cuda", generator=gen)) for _ in range(2)]
    noise_sh = [torch.view_as_complex(torch.randn(B, S, wl.n_sh, 3, 3, 2, device="cuda", generator=gen)) for _ in range(2)]
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, wl.n_sh, 3, 3), dtype=torch.complex64, device="cuda")
    cn2, dz = list(wl.cn2_list), list(wl.dz)
    ssp.make_screens(N, wl.dx, pg, wl.lam, cn2, dz, wl.n_sh, noise[0], noise_sh[0], spectrum=spec, sh_coef=shc)
    # as bench.py does it: the frame's fresh grid noise is drawn inside the generator (ssp_evolve_screens_seeded); the same
    # draws are written out by ssp_fill_noise for the oracle (tests/test_gpu_noise.py: the two are the same bytes)
    ssp.fill_noise(1234, 2, noise[1])
    scr = ssp.evolve_screens_seeded(N, wl.dx, pg, wl.lam, cn2, dz, wl.n_sh, wl.ar_a, 0, 0, 0, 1234, 2, 0, noise_sh[1], spec, shc)
    # the oracle consumes the same white noise (as drawn on the device, copied back) for realisation b_s
    f2 = lambda t: np.ascontiguousarray(torch.view_as_real(t[b_s:b_s + 1]).cpu().numpy())
    _, spec_ref, shc_ref = orc.make_screens(N, wl.dx, po, wl.lam, wl.cn2_list, wl.dz, wl.n_sh, f2(noise[0]), f2(noise_sh[0]))
    scr_ref = orc.evolve_screens(N, wl.dx, po, wl.lam, wl.cn2_list, wl.dz, wl.n_sh, wl.ar_a, 0, 0, 0, f2(noise[1]),
                                 f2(noise_sh[1]), spec_ref, shc_ref)
    assert rel_l2(scr[b_s:b_s + 1].cpu().numpy(), scr_ref).max() < tol(N, 2)
    u0 = synth.input_field(wl, B)
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    out = ssp.propagate(N, wl.dx, wl.lam, dz, cu(u0), scr, stats=stats, roi_frac=0.25, **kw)
    gin = ssp.propagate_adjoint(N, wl.dx, wl.lam, dz, out, scr, **kw)
    scr32 = scr[b_s:b_s + 1].cpu().numpy()                    # the GPU's own fp32 screens of that realisation
    ref = orc.propagate(N, wl.dx, wl.lam, wl.dz, u0[b_s:b_s + 1], scr32, **kw)
    assert rel_l2(out[b_s:b_s + 1].cpu().numpy(), ref).max() < tol(N, S)
    gref = orc.propagate_adjoint(N, wl.dx, wl.lam, wl.dz, out[b_s:b_s + 1].cpu().numpy(), scr32, **kw)
    assert rel_l2(gin[b_s:b_s + 1].cpu().numpy(), gref).max() < tol(N, S)
    _check_stats(api.stats_to_dicts(stats)[b_s:b_s + 1], orc.beam_stats(N, wl.dx, ref, roi_frac=0.25), wl)
    # any size: <A x, y> = <x, A^H y> per realisation with y = A x, and power never grows (|H| = 1, |W| <= 1)
    ip1 = ssp.inner_products(N, wl.dx, out, out).cpu().numpy()          # <Ax, Ax>
    ip2 = ssp.inner_products(N, wl.dx, gin, cu(u0)).cpu().numpy()       # <A^H A x, x>
    p0 = ssp.inner_products(N, wl.dx, cu(u0), cu(u0)).cpu().numpy()[:, 2]
    for b in range(B):
        assert abs(ip1[b, 0] - ip2[b, 0]) < 2e-6 * S * ip1[b, 0], (b, ip1[b], ip2[b])
        assert abs(ip2[b, 1]) < 2e-6 * S * ip1[b, 0]
        assert ip1[b, 2] <= p0[b] * (1 + 1e-5)
    # distinct noise per realisation gives distinct fields; all finite
    assert torch.isfinite(torch.view_as_real(out)).all()
    assert not torch.equal(out[0], out[1])


@pytest.mark.parametrize("cid", [2, 4, 5])
def test_full_size_configs_properties(ssp, cid):
    """configs[1], [3], [4] at their FULL sizes (512^2 x 64 x 10, 2048^2 x 8 x 30, 4096^2 x 2 x 20): too large for the
    fp64 oracle, so what is checked are properties that hold at any size -- finite output, power never grows
    (|H| = 1, |W| <= 1, |exp(i phi)| = 1), <A x, A x> = <A^H A x, x> per realisation, piston-free screens -- on
    screens generated on the device from seeded noise."""
    import torch
    from paper_2604_07248_b200 import api
    wl = synth.CONFIGS[cid]
    N, S, B = wl.N, wl.S, wl.B
    pg = api.PsdParams(**wl.psd_dict())
    gen = torch.Generator(device="cuda")
    gen.manual_seed(100 + cid)
    noise = torch.view_as_complex(torch.randn(B, S, N, N, 2, device="cuda", generator=gen))
    nsh = torch.view_as_complex(torch.randn(B, S, max(wl.n_sh, 1), 3, 3, 2, device="cuda", generator=gen))
    cn2 = list(wl.cn2_list) if cid != 2 else [wl.cn2_sweep[1]] * S
    scr = ssp.make_screens(N, wl.dx, pg, wl.lam, cn2, list(wl.dz), wl.n_sh, noise, nsh if wl.n_sh else None)
    del noise
    assert torch.isfinite(scr).all()
    m = scr.mean(dim=(-2, -1)).abs().max()
    assert float(m) < 1e-3 * float(scr.abs().max())
    u0 = cu(synth.input_field(wl, B))
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    out = ssp.propagate(N, wl.dx, wl.lam, list(wl.dz), u0, scr, **kw)
    gin = ssp.propagate_adjoint(N, wl.dx, wl.lam, list(wl.dz), out, scr, **kw)
    assert torch.isfinite(torch.view_as_real(out)).all()
    ip1 = ssp.inner_products(N, wl.dx, out, out).cpu().numpy()
    ip2 = ssp.inner_products(N, wl.dx, gin, u0).cpu().numpy()
    p0 = ssp.inner_products(N, wl.dx, u0, u0).cpu().numpy()[:, 2]
    for b in range(B):
        assert abs(ip1[b, 0] - ip2[b, 0]) < 2e-6 * S * ip1[b, 0], (b, ip1[b], ip2[b])
        assert abs(ip2[b, 1]) < 2e-6 * S * ip1[b, 0]
        assert ip1[b, 2] <= p0[b] * (1 + 1e-5)


@pytest.mark.parametrize("n_sh,wind", [(3, False), (2, True), (0, False)])
def test_fused_screen_synthesis_frame(ssp, orc, n_sh, wind):
    """ssp_evolve_propagate (the generator's row pass fused into the split step's row kernel, forward-only
    temporal frames at 1024^2): two successive AR frames of 3 stacks x 4 von Karman screens.  Against the oracle
    (evolve_screens + propagate on the same noise), against the unfused GPU calls (same AR state bit for bit, fields to
    fp32 rounding), statistics included; odd batch, wind, with and without subharmonics."""
    import torch
    from paper_2604_07248_b200 import api
    wl = synth.CONFIGS[3]
    N, S, B = wl.N, 4, 3
    po, pg = _psd(wl, orc)
    cn2, dz = list(wl.cn2_list[:S] * np.array([1.0, 2.0, 0.5, 1.5])), list(wl.dz[:S] * np.array([1.0, 0.7, 1.3, 1.0]))
    a, T = 0.97, 0.01
    vx, vy = (2.3 * wl.dx / T, -0.7 * wl.dx / T) if wind else (0.0, 0.0)
    frames = [synth.noise(33, n_sh, b, S, N, n_sh, frames=3) for b in range(B)]
    hi = lambda t: np.stack([frames[b][t][0] for b in range(B)])
    sh = lambda t: np.stack([frames[b][t][1] for b in range(B)])
    _, spec_ref, shc_ref = oracle_screens_parallel(orc, N, wl.dx, po, wl.lam, cn2, dz, n_sh, hi(0), sh(0), keep_spectrum=True)
    spec_ref = np.ascontiguousarray(spec_ref)
    shc_ref = np.ascontiguousarray(shc_ref) if n_sh else None
    spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    shc = torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device="cuda")
    ssp.make_screens(N, wl.dx, pg, wl.lam, cn2, dz, n_sh, cu(c64(hi(0))), cu(c64(sh(0))) if n_sh else None,
                     spectrum=spec, sh_coef=shc if n_sh else None)
    spec_u, shc_u = spec.clone(), shc.clone()                       # the unfused GPU path's AR state
    ycol = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    u0 = synth.input_field(wl, B)
    kw = dict(win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    for t in (1, 2):
        h_t, s_t = hi(t), sh(t)
        d_h, d_s = cu(c64(h_t)), (cu(c64(s_t)) if n_sh else None)
        stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        l0 = ssp.launch_count()
        out = ssp.evolve_propagate(N, wl.dx, pg, wl.lam, cn2, dz, n_sh, a, vx, vy, T, d_h, d_s, spec, shc if n_sh else None,
                                   cu(u0), ycol, stats=stats, roi_frac=0.25, **kw)
        n_fused = ssp.launch_count() - l0
        # unfused GPU path
        scr_u = ssp.evolve_screens(N, wl.dx, pg, wl.lam, cn2, dz, n_sh, a, vx, vy, T, d_h, d_s, spec_u, shc_u if n_sh else None)
        stats_u = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        out_u = ssp.propagate(N, wl.dx, wl.lam, dz, cu(u0), scr_u, stats=stats_u, roi_frac=0.25, **kw)
        assert torch.equal(spec, spec_u) and torch.equal(shc, shc_u)
        e_gpu = rel_l2(out.cpu().numpy(), out_u.cpu().numpy().astype(np.complex128)).max()
        assert e_gpu < 2e-6 * S, e_gpu
        # oracle
        def evolve_one(bs):
            b, j = divmod(bs, S)
            sp = np.ascontiguousarray(spec_ref[b:b + 1, j:j + 1])
            sc = np.ascontiguousarray(shc_ref[b:b + 1, j:j + 1]) if n_sh else None
            o = orc.evolve_screens(N, wl.dx, po, wl.lam, [cn2[j]], [dz[j]], n_sh, a, vx, vy, T, h_t[b:b + 1, j:j + 1],
                                   s_t[b:b + 1, j:j + 1] if n_sh else None, sp, sc)
            return o[0, 0], sp[0, 0], (sc[0, 0] if n_sh else None)
        res = pmap(evolve_one, range(B * S))
        scr_ref = np.stack([r[0] for r in res]).reshape(B, S, N, N)
        spec_ref = np.stack([r[1] for r in res]).reshape(B, S, N, N)
        if n_sh:
            shc_ref = np.stack([r[2] for r in res]).reshape(B, S, n_sh, 3, 3)
        # the oracle propagates through ITS fp64 screens: the fused path never rounds a screen to fp32 in memory
        ref = np.concatenate(pmap(lambda b: orc.propagate(N, wl.dx, wl.lam, dz, u0[b:b + 1], scr_ref[b:b + 1], **kw), range(B)))
        e_f = rel_l2(out.cpu().numpy(), ref).max()
        record("fused_frame", n_sh=n_sh, wind=wind, frame=t, vs_unfused=float(e_gpu), field=float(e_f), bound=tol(N, S + t + 1),
               launches=int(n_fused))
        assert e_f < tol(N, S + t + 1), (t, e_f)
        _check_stats(api.stats_to_dicts(stats), orc.beam_stats(N, wl.dx, ref, roi_frac=0.25), wl)
    # argument errors: other grids are refused, not silently run unfused
    with pytest.raises(api.SspError) as ei:
        small = torch.zeros((1, 1, 512, 512), dtype=torch.complex64, device="cuda")
        ssp.evolve_propagate(512, wl.dx, pg, wl.lam, [cn2[0]], [dz[0]], 0, a, 0, 0, 0, small, None, small.clone(), None,
                             small[0].clone(), small.clone(), **kw)
    assert ei.value.code == api.EUNSUPPORTED
