"""GPU parity: split-step propagation, adjoint and statistics through the C ABI vs the CPU oracle.

Bar (BASELINE.json north_star): per-field relative L2 error <= 2e-5 * log2(N) * screens."""
import math

import numpy as np
import pytest

from paper_2604_07248_b200 import synth
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


def tol(N, n_screens):
    return 2e-5 * math.log2(N) * max(1, n_screens)


def _case(N, B, n_steps, S, seed):
    dx, lam = 1e-3, 1.0e-6
    rng = np.random.default_rng(seed)
    # steps of the order of the aliasing-free distance N dx^2 / lambda, uneven on purpose
    dz = (N * dx * dx / lam) * (0.1 + 0.3 * rng.random(n_steps))
    u0 = synth.random_field(N, B, seed)
    scr = synth.random_screens(N, B, max(S, 1), seed, rms=3.0)[:, :S]
    return dx, lam, dz, u0, scr


@pytest.mark.parametrize("N", [8, 16, 32, 64, 128, 256, 512, 1024])
def test_propagate_parity_all_plans(ssp, orc, N):
    """Every FFT plan (1, 2 stages), per-realisation screens, window on, uneven dz."""
    B, n_steps, S = (3, 3, 3) if N <= 512 else (2, 2, 2)
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, N)
    ref = orc.propagate(N, dx, lam, dz, u0, scr, win_order=16, win_sigma_frac=0.47)
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), win_order=16, win_sigma_frac=0.47)
    err = rel_l2(out.cpu().numpy(), ref)
    assert err.max() < tol(N, S), err
    assert err.max() < 5e-6 * n_steps + 1e-6, err        # what fp32 actually delivers


@pytest.mark.parametrize("N", [2048, 4096])
def test_propagate_parity_three_stage_plans(ssp, orc, N):
    B, n_steps, S = 1, 2, 2
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, N)
    ref = orc.propagate(N, dx, lam, dz, u0, scr, win_order=16, win_sigma_frac=0.47)
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), win_order=16, win_sigma_frac=0.47)
    err = rel_l2(out.cpu().numpy(), ref)
    assert err.max() < tol(N, S), err


def test_propagate_variants(ssp, orc):
    """In place, shared stack, trailing vacuum step (S = n_steps - 1), no window, n0, planes."""
    import torch
    N, B, n_steps = 64, 3, 4
    dx, lam, dz, u0, scr = _case(N, B, n_steps, 3, 7)
    # shared stack + trailing vacuum step + refractive index
    ref = orc.propagate(N, dx, lam, dz, u0, scr[0], shared_screens=True, n0=1.33)
    d = cu(u0)
    out = ssp.propagate(N, dx, lam, list(dz), d, cu(scr[0]), shared_screens=True, n0=1.33, out=d)  # in place
    assert out.data_ptr() == d.data_ptr()
    assert rel_l2(out.cpu().numpy(), ref).max() < tol(N, 3)
    # vacuum only (S = 0)
    ref = orc.propagate(N, dx, lam, dz, u0)
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0))
    assert rel_l2(out.cpu().numpy(), ref).max() < tol(N, 1)
    # saved planes = field after every complete step
    ref, ref_planes = orc.propagate(N, dx, lam, dz, u0, scr, win_order=8, win_sigma_frac=0.45, return_planes=True)
    planes = torch.empty((B, n_steps, N, N), dtype=torch.complex64, device="cuda")
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), win_order=8, win_sigma_frac=0.45, planes=planes)
    assert rel_l2(planes.cpu().numpy(), ref_planes).max() < tol(N, 3)
    assert torch.equal(planes[:, -1], out)


def test_config1_full(ssp, orc):
    """BASELINE.json configs[0] in full: 128^2, 5 von Karman screens + 3 subharmonic levels, 4 realisations,
    Gaussian beam, super-Gaussian window; received field, beam width, scintillation index."""
    from paper_2604_07248_b200 import api
    wl = synth.CONFIGS[1]
    N, B, S = wl.N, wl.B, wl.S
    hi, sh = synth.noise_batch(1, 0, B, S, N, wl.n_sh)
    psd_o = orc.Psd(**wl.psd_dict())
    scr_ref, _, _ = orc.make_screens(N, wl.dx, psd_o, wl.lam, wl.cn2_list, wl.dz, wl.n_sh, hi, sh)
    scr32 = scr_ref.astype(np.float32)                       # the same fp32 screens feed both sides
    u0 = synth.input_field(wl)
    ref = orc.propagate(N, wl.dx, wl.lam, wl.dz, u0, scr32, win_order=wl.win_order, win_sigma_frac=wl.win_sigma_frac)
    import torch
    stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    out = ssp.propagate(N, wl.dx, wl.lam, list(wl.dz), cu(u0), cu(scr32), win_order=wl.win_order,
                        win_sigma_frac=wl.win_sigma_frac, stats=stats, roi_frac=0.25)
    err = rel_l2(out.cpu().numpy(), ref)
    assert err.max() < tol(N, S), err
    st_ref = orc.beam_stats(N, wl.dx, ref, roi_frac=0.25)
    st = api.stats_to_dicts(stats)
    for a, b in zip(st, st_ref):
        for k in ("power", "w2", "sxx", "syy", "roi_sumI", "roi_sumI2", "I_axis"):
            assert abs(a[k] / b[k] - 1) < 1e-4, (k, a[k], b[k])
        assert abs(a["cx"] - b["cx"]) < 1e-4 * wl.dx * N and abs(a["cy"] - b["cy"]) < 1e-4 * wl.dx * N
        assert abs(a["sxy"] - b["sxy"]) < 1e-4 * (b["sxx"] + b["syy"])
        assert a["roi_n"] == b["roi_n"]


@pytest.mark.parametrize("N,dx,lam", [(64, 0.6e-6, 1.0e-6), (256, 2e-6, 1.0e-6), (512, 0.7e-6, 1.0e-6), (512, 1e-3, 1.0e-6),
                                      (1024, 1e-3, 1.0e-6), (2048, 1e-3, 1.0e-6), (4096, 1e-3, 1.0e-6)])
def test_angular_spectrum_parity(ssp, orc, N, dx, lam):
    """Angular-spectrum H (Eq.6, carrier removed): non-paraxial grids with evanescent corner bins
    (dx < lambda) through the register-load column kernel, paraxial ones through the TMA kernel; forward,
    adjoint, and the adjoint identity."""
    from paper_2604_07248_b200 import api
    B, n_steps, S = (2, 3, 2) if N <= 1024 else ((1, 2, 2) if N == 2048 else (1, 1, 1))
    rng = np.random.default_rng(N)
    dz = (N * dx * dx / lam) * (0.1 + 0.3 * rng.random(n_steps))
    u0 = synth.random_field(N, B, N + 1)
    scr = synth.random_screens(N, B, S, N + 2, rms=2.0)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    ref = orc.propagate(N, dx, lam, dz, u0, scr, h_kind=orc.H_ANGULAR_SPECTRUM, n0=1.1, **kw)
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), h_kind=api.H_ANGULAR_SPECTRUM, n0=1.1, **kw)
    assert rel_l2(out.cpu().numpy(), ref).max() < tol(N, S)
    if dx < lam:                                              # the two kernels differ here (and bins are cut)
        fres = orc.propagate(N, dx, lam, dz, u0, scr, n0=1.1, **kw)
        assert rel_l2(ref, fres).min() > 0.1
    g = synth.random_field(N, B, N + 3)
    gref = orc.propagate_adjoint(N, dx, lam, dz, g, scr, h_kind=orc.H_ANGULAR_SPECTRUM, n0=1.1, **kw)
    gin = ssp.propagate_adjoint(N, dx, lam, list(dz), cu(g), cu(scr), h_kind=api.H_ANGULAR_SPECTRUM, n0=1.1, **kw)
    assert rel_l2(gin.cpu().numpy(), gref).max() < tol(N, S)
    ip1 = ssp.inner_products(N, dx, cu(g), out).cpu().numpy()       # <g, A u0>
    ip2 = ssp.inner_products(N, dx, gin, cu(u0)).cpu().numpy()      # <A^H g, u0>
    for b in range(B):
        scale = math.sqrt(ip1[b, 2] * ip1[b, 3])
        assert abs(complex(ip1[b, 0], ip1[b, 1]) - complex(ip2[b, 0], ip2[b, 1])) < 2e-6 * n_steps * scale


def test_adjoint_parity_and_gradient(ssp, orc):
    import torch
    N, B, n_steps, S = 64, 2, 4, 3
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, 21)
    kw = dict(win_order=8, win_sigma_frac=0.45)
    out_ref, planes_ref = orc.propagate(N, dx, lam, dz, u0, scr, return_planes=True, **kw)
    g_out = synth.random_field(N, B, 22)
    gin_ref, grad_ref = orc.propagate_adjoint(N, dx, lam, dz, g_out, scr, planes=planes_ref.astype(np.complex64), **kw)
    planes = cu(planes_ref.astype(np.complex64))
    grad = torch.zeros((B, S, N, N), dtype=torch.float32, device="cuda")
    gin = ssp.propagate_adjoint(N, dx, lam, list(dz), cu(g_out), cu(scr), planes=planes, phase_grad=grad, **kw)
    assert rel_l2(gin.cpu().numpy(), gin_ref).max() < tol(N, S)
    gerr = rel_l2(grad.cpu().numpy(), grad_ref)
    assert gerr.max() < tol(N, S + 2), gerr
    # without gradient outputs, in place
    d = cu(g_out)
    gin2 = ssp.propagate_adjoint(N, dx, lam, list(dz), d, cu(scr), out=d, **kw)
    assert rel_l2(gin2.cpu().numpy(), gin_ref).max() < tol(N, S)


@pytest.mark.parametrize("N,shared", [(1024, False), (1024, True), (512, False)])
def test_phase_gradient_generic_row_kernel_headline_grid(ssp, orc, N, shared):
    """d_phase_grad = Im(G_j conj(U_j)) (O7) at the headline grid against the oracle: at 1024^2 the saved
    planes and the gradient go through the GENERIC row kernel, which reads the column kernel's re/im-swapped hand-over
    behind a run-time flag and the cached window map through a run-time pointer (round 1 only checked isfinite there).
    Trailing vacuum step (S = n_steps - 1), per-field and shared screen stacks; a sign, swap or stride error in the
    epilogue shows as an O(1) relative error."""
    import torch
    B, n_steps, S = 2, 3, 2
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, 900 + N)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    scr_o = scr[0] if shared else scr
    out_ref, planes_ref = orc.propagate(N, dx, lam, dz, u0, scr_o, shared_screens=shared, return_planes=True, **kw)
    planes = torch.empty((B, n_steps, N, N), dtype=torch.complex64, device="cuda")
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr_o), shared_screens=shared, planes=planes, **kw)
    assert rel_l2(out.cpu().numpy(), out_ref).max() < tol(N, S)
    assert rel_l2(planes.cpu().numpy(), planes_ref).max() < tol(N, S)
    g_out = synth.random_field(N, B, 901 + N)
    # the oracle's gradient on the GPU's own (fp32) planes: isolates the adjoint + epilogue
    p32 = planes.cpu().numpy()
    gin_ref, grad_ref = orc.propagate_adjoint(N, dx, lam, dz, g_out, scr_o, shared_screens=shared, planes=p32, **kw)
    grad = torch.full((B, S, N, N), float("nan"), dtype=torch.float32, device="cuda")
    gin = ssp.propagate_adjoint(N, dx, lam, list(dz), cu(g_out), cu(scr_o), shared_screens=shared, planes=planes,
                                phase_grad=grad, **kw)
    assert rel_l2(gin.cpu().numpy(), gin_ref).max() < tol(N, S)
    gerr = rel_l2(grad.cpu().numpy(), grad_ref)
    assert gerr.max() < tol(N, S + 2), gerr
    from tests.util import record
    record("phase_grad", N=N, shared=shared, grad=float(gerr.max()), bound=tol(N, S + 2))
    # the gradient means what it says: d/d phi of Re<g_out, A(u0)> by central differences at a few pixels of screen 1
    if not shared:
        b, j = 1, 0
        base = scr.copy()
        for (iy, ix) in [(N // 2, N // 2), (N // 2 + 3, N // 2 - 5), (N // 3, N // 2 + 7)]:
            vals = []
            for e in (+1e-2, -1e-2):
                pert = base.copy()
                pert[b, j, iy, ix] += e
                o = orc.propagate(N, dx, lam, dz, u0[b:b + 1], pert[b:b + 1], **kw)
                vals.append(np.real(np.vdot(g_out[b].astype(np.complex128), o[0])))
            fd = (vals[0] - vals[1]) / 2e-2
            got = float(grad[b, j, iy, ix])
            assert abs(got - fd) < 2e-3 * max(abs(fd), np.abs(grad_ref[b, j]).max() * 0.05), (iy, ix, got, fd)


@pytest.mark.parametrize("N", [32, 256, 1024])
def test_adjoint_identity_on_gpu(ssp, N):
    """<A x, y> = <x, A^H y> evaluated entirely on the GPU path (a property that holds at any size)."""
    B, n_steps, S = 2, 3, 3
    dx, lam, dz, x, scr = _case(N, B, n_steps, S, 31)
    y = synth.random_field(N, B, 32)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    Ax = ssp.propagate(N, dx, lam, list(dz), cu(x), cu(scr), **kw)
    AHy = ssp.propagate_adjoint(N, dx, lam, list(dz), cu(y), cu(scr), **kw)
    ip1 = ssp.inner_products(N, dx, cu(y), Ax).cpu().numpy()       # <y, A x>
    ip2 = ssp.inner_products(N, dx, AHy, cu(x)).cpu().numpy()      # <A^H y, x>
    for b in range(B):
        lhs = complex(ip1[b, 0], ip1[b, 1])
        rhs = complex(ip2[b, 0], ip2[b, 1])
        scale = math.sqrt(ip1[b, 2] * ip1[b, 3])
        assert abs(lhs - rhs) < 2e-6 * n_steps * scale, (lhs, rhs)


def test_beam_stats_and_welford(ssp, orc):
    import torch
    from paper_2604_07248_b200 import api
    N, dx, B = 128, 2e-3, 5
    rng = np.random.default_rng(3)
    x = synth.coords(N, dx)
    X, Y = np.meshgrid(x, x)
    fields = []
    for b in range(B):
        x0, y0, wx, wy = rng.normal(0, 0.02), rng.normal(0, 0.02), 0.02 + 0.02 * rng.random(), 0.02 + 0.02 * rng.random()
        fields.append(np.exp(-((X - x0) / wx) ** 2 - ((Y - y0) / wy) ** 2 + 1j * rng.random() * X * 30))
    u = (np.stack(fields) + 0.01 * synth.random_field(N, B, 5)).astype(np.complex64)
    for roi in (0.0, 0.3, 1.0):
        st_ref = orc.beam_stats(N, dx, u, roi_frac=roi)
        stats, _ = ssp.beam_stats(N, dx, cu(u), roi_frac=roi)
        for a, r in zip(api.stats_to_dicts(stats), st_ref):
            for k in ("power", "w2", "sxx", "syy", "I_axis", "roi_sumI", "roi_sumI2"):
                assert abs(a[k] / r[k] - 1) < 1e-6, (roi, k, a[k], r[k])
            for k in ("cx", "cy"):
                assert abs(a[k] - r[k]) < 1e-7 * dx * N
            assert abs(a["sxy"] - r["sxy"]) < 1e-6 * (r["sxx"] + r["syy"])
            assert a["roi_n"] == r["roi_n"]
    mean = torch.zeros((N, N), dtype=torch.float32, device="cuda")
    M2 = torch.zeros((N, N), dtype=torch.float32, device="cuda")
    _, cnt = ssp.beam_stats(N, dx, cu(u[:2]), mean=mean, M2=M2, count=0)
    _, cnt = ssp.beam_stats(N, dx, cu(u[2:]), mean=mean, M2=M2, count=cnt)
    m_ref, M2_ref = np.zeros((N, N)), np.zeros((N, N))
    c_ref = orc.welford(N, u, m_ref, M2_ref, 0)
    assert cnt == c_ref == B
    np.testing.assert_allclose(mean.cpu().numpy(), m_ref, rtol=2e-5, atol=1e-7)
    np.testing.assert_allclose(M2.cpu().numpy(), M2_ref, rtol=2e-4, atol=1e-7)


@pytest.mark.parametrize("N", [8, 16, 32, 64])
def test_beam_stats_small_grids(ssp, orc, N):
    """Grids with fewer rows than one pass of the reducer (N = 8, 16: a host-side division by zero in round 1), through
    ssp_beam_stats and through ssp_propagate's statistics epilogue, B = 1, 4 and a batch beyond one wave."""
    from paper_2604_07248_b200 import api
    dx = 1e-3
    for B in (1, 4, 300):
        u = (synth.random_field(N, B, 100 + N) + synth.gaussian_beam(N, dx, 0.2 * N * dx, B)).astype(np.complex64)
        for roi in (0.0, 0.5, 1.0):
            st_ref = orc.beam_stats(N, dx, u, roi_frac=roi)
            stats, _ = ssp.beam_stats(N, dx, cu(u), roi_frac=roi)
            for a, r in zip(api.stats_to_dicts(stats), st_ref):
                for k in ("power", "w2", "sxx", "syy", "I_axis", "roi_sumI", "roi_sumI2"):
                    assert abs(a[k] / r[k] - 1) < 1e-6, (B, roi, k, a[k], r[k])
                assert abs(a["cx"] - r["cx"]) < 1e-7 * dx * N and abs(a["cy"] - r["cy"]) < 1e-7 * dx * N
                assert a["roi_n"] == r["roi_n"]
    import torch
    B = 3
    dx, lam, dz, u0, scr = _case(N, B, 2, 2, 7 * N)
    stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), win_order=16, win_sigma_frac=0.47, stats=stats, roi_frac=0.5)
    ref = orc.propagate(N, dx, lam, dz, u0, scr, win_order=16, win_sigma_frac=0.47)
    for a, r in zip(api.stats_to_dicts(stats), orc.beam_stats(N, dx, ref, roi_frac=0.5)):
        for k in ("power", "w2", "I_axis", "roi_sumI", "roi_sumI2"):
            assert abs(a[k] / r[k] - 1) < 1e-4, (k, a[k], r[k])


@pytest.mark.parametrize("N", [8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096])
def test_statistics_epilogue_of_the_last_row_kernel(ssp, orc, N):
    """K8 rides on the last row pass (fused, 0 B/px): ssp_propagate(..., d_stats) launches no stand-alone
    reducer -- one finaliser launch on top of the propagation (none on the on-chip path) -- and the records equal those
    of ssp_beam_stats on the returned field (same pixels, different summation order: 1e-6) and the oracle's (1e-4).
    Odd batch, per-field screens, trailing vacuum step, and the planes-saving generic kernel as well."""
    import torch
    from paper_2604_07248_b200 import api
    B, n_steps, S = (3, 3, 2) if N <= 1024 else (1, 2, 2)
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, 5000 + N)
    u0 = (u0 + 3.0 * synth.gaussian_beam(N, dx, 0.15 * N * dx, B)).astype(np.complex64)   # a beam over noise: nontrivial moments
    kw = dict(win_order=16, win_sigma_frac=0.47)
    ref = orc.propagate(N, dx, lam, dz, u0, scr, **kw) if N <= 1024 else None
    ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), **kw)          # first use builds cached tables (window map)
    for roi, with_planes in ((0.25, False), (0.0, False), (1.0, True)):
        stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        planes = torch.empty((B, n_steps, N, N), dtype=torch.complex64, device="cuda") if with_planes else None
        l0 = ssp.launch_count()
        out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), stats=stats, roi_frac=roi, planes=planes, **kw)
        n_launch = ssp.launch_count() - l0
        single_cta = N == 64 and not with_planes                   # statistics finished inside the kernel
        cluster = N == 128 and not with_planes                     # one cluster launch + the finaliser
        assert n_launch == (1 if single_cta else (2 if cluster else 2 * n_steps + 1 + 1)), n_launch
        got = api.stats_to_dicts(stats)
        alone, _ = ssp.beam_stats(N, dx, out, roi_frac=roi)
        for a, r in zip(got, api.stats_to_dicts(alone)):
            for k in ("power", "w2", "sxx", "syy", "I_axis", "roi_sumI", "roi_sumI2"):
                assert abs(a[k] / r[k] - 1) < 1e-6, (roi, k, a[k], r[k])
            assert abs(a["cx"] - r["cx"]) < 1e-7 * dx * N and abs(a["cy"] - r["cy"]) < 1e-7 * dx * N
            assert abs(a["sxy"] - r["sxy"]) < 1e-6 * (r["sxx"] + r["syy"])
            assert a["roi_n"] == r["roi_n"]
        if ref is not None:
            for a, r in zip(got, orc.beam_stats(N, dx, ref, roi_frac=roi)):
                for k in ("power", "w2", "I_axis", "roi_sumI", "roi_sumI2"):
                    assert abs(a[k] / r[k] - 1) < 1e-4, (roi, k, a[k], r[k])
                assert a["roi_n"] == r["roi_n"]


def test_transfer_table_cache_overflow_keeps_pointers_valid(ssp, orc):
    """The context caches one 1-D transfer-function table per distinct (N, dx, lambda, dz, conj, scaled) and drops the
    cache beyond 4096 entries -- at the entry of a call only, never between the look-ups of one call (round 1 freed
    tables the on-chip path had already collected).  Fill the cache past the cap with throw-away steps, then run an
    N = 128 stack of distinct steps (on-chip path: all tables gathered before the one launch) against the oracle."""
    N, B, n_steps = 128, 2, 6
    dx, lam, dz, u0, scr = _case(N, B, n_steps, n_steps, 4242)
    ref = orc.propagate(N, dx, lam, dz, u0, scr, win_order=16, win_sigma_frac=0.47)
    d_u0, d_scr = cu(u0), cu(scr)
    small = cu(synth.random_field(8, 1, 1))
    for rep in range(3):
        for chunk in range(9):                                     # 9 x 240 steps x 2 tables each > 4096 per repetition
            dzs = [1.0 + 1e-3 * (rep * 10000 + chunk * 240 + j) for j in range(240)]
            ssp.propagate(8, dx, lam, dzs, small, None)
        out = ssp.propagate(N, dx, lam, list(dz), d_u0, d_scr, win_order=16, win_sigma_frac=0.47)
        err = rel_l2(out.cpu().numpy(), ref)
        assert err.max() < tol(N, n_steps), (rep, err)
        g = ssp.propagate_adjoint(N, dx, lam, list(dz), out, d_scr, win_order=16, win_sigma_frac=0.47)
        gref = orc.propagate_adjoint(N, dx, lam, dz, out.cpu().numpy(), scr, win_order=16, win_sigma_frac=0.47)
        assert rel_l2(g.cpu().numpy(), gref).max() < tol(N, n_steps)


def test_error_codes(ssp):
    import torch
    from paper_2604_07248_b200 import api
    N, dx, lam = 64, 1e-3, 1e-6
    u = torch.zeros((1, N, N), dtype=torch.complex64, device="cuda")
    scr = torch.zeros((1, 2, N, N), dtype=torch.float32, device="cuda")
    with pytest.raises(api.SspError) as e:
        ssp.propagate(48, dx, lam, [1.0], torch.zeros((1, 48, 48), dtype=torch.complex64, device="cuda"))
    assert e.value.code == api.EINVAL
    with pytest.raises(api.SspError) as e:
        ssp.propagate(N, dx, lam, [1.0], u, scr)                  # S = 2 > n_steps = 1
    assert e.value.code == api.EINVAL
    with pytest.raises(api.SspError) as e:
        ssp.propagate(N, dx, lam, [1.0, -2.0], u)
    assert e.value.code == api.EINVAL
    with pytest.raises(api.SspError) as e:
        ssp.propagate(N, dx, lam, [1.0], u, h_kind=7)
    assert e.value.code == api.EINVAL
    with pytest.raises(api.SspError) as e:
        ssp.propagate(N, dx, -1.0, [1.0], u)
    assert e.value.code == api.EINVAL
    with pytest.raises(api.SspError) as e:                        # empty batch
        ssp.propagate(N, dx, lam, [1.0], torch.zeros((0, N, N), dtype=torch.complex64, device="cuda"))
    assert e.value.code == api.EINVAL
    with pytest.raises(api.SspError) as e:                        # no steps
        ssp.propagate(N, dx, lam, [], u)
    assert e.value.code == api.EINVAL
    with pytest.raises(TypeError):
        ssp.propagate(N, dx, lam, [1.0], u.cpu())                # no CPU fallback
    assert ssp.launch_count() >= 0


@pytest.mark.parametrize("B,shared", [(1, False), (11, False), (16, True)])
def test_propagate_host_matches_device_path(ssp, orc, B, shared):
    """ssp_propagate_host (host buffers, chunked copy/compute pipeline) returns exactly what ssp_propagate returns on
    the same inputs, and one field is checked against the oracle."""
    import torch
    from paper_2604_07248_b200 import api
    N, n_steps, S = 128, 3, 3
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, 100 + B)
    if shared:
        scr = scr[0]
    kw = dict(win_order=16, win_sigma_frac=0.47)
    stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    ref_dev = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), shared_screens=shared, stats=stats, roi_frac=0.5, **kw)
    h_in = torch.from_numpy(u0).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    h_scr = torch.from_numpy(np.ascontiguousarray(scr)).pin_memory()
    h_st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8).pin_memory()
    d_field = torch.empty((B, N, N), dtype=torch.complex64, device="cuda")
    d_scr = torch.empty(scr.shape, dtype=torch.float32, device="cuda")
    d_st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    ssp.propagate_host(N, dx, lam, list(dz), h_in, h_out, h_scr, shared, S, 16, 0.47, h_st, 0.5, d_field, d_scr, d_st)
    assert torch.equal(h_out, ref_dev.cpu())
    # screens already on the device (h_screens = None): only the fields travel, same result
    h_out2 = torch.empty_like(h_in).pin_memory()
    ssp.propagate_host(N, dx, lam, list(dz), h_in, h_out2, None, shared, S, 16, 0.47, h_st, 0.5, d_field, cu(scr), d_st)
    assert torch.equal(h_out2, h_out)
    for a, b in zip(api.stats_to_dicts(h_st), api.stats_to_dicts(stats)):   # chunks group the fp64 partial sums differently
        for k in ("power", "w2", "sxx", "syy", "roi_sumI", "roi_sumI2", "I_axis"):
            assert abs(a[k] / b[k] - 1) < 1e-12, (k, a[k], b[k])
        assert a["roi_n"] == b["roi_n"]
    ref = orc.propagate(N, dx, lam, dz, u0[-1:], scr if shared else scr[-1:], shared_screens=shared, **kw)
    assert rel_l2(h_out[-1:].numpy(), ref).max() < tol(N, S)


@pytest.mark.parametrize("N", [64, 1024])
def test_aperture_bit_exact(ssp, orc, N):
    """Circular aperture: an integer decision, so the mask is compared exactly."""
    dx, B = 0.34e-3, 2
    u = synth.random_field(N, B, 70 + N)
    for R in (0.0, 0.3048 / 2 * N / 1024, 0.37 * N * dx, 10.0):
        ref = orc.aperture(N, dx, R, u)
        d = cu(u)
        out = ssp.aperture(N, dx, R, d)
        np.testing.assert_array_equal(out.cpu().numpy(), ref.astype(np.complex64))
        ssp.aperture(N, dx, R, d, out=d)                      # in place
        np.testing.assert_array_equal(d.cpu().numpy(), ref.astype(np.complex64))


@pytest.mark.parametrize("N,B", [(64, 5), (128, 5), (128, 64), (128, 70)])
def test_on_chip_path_matches_multi_kernel_path(ssp, orc, N, B):
    """Small grids without saved planes run the whole stack in ONE launch with the field resident in shared memory:
    one CTA per field (ssp_small.cu: N = 64, and N = 128 at batches beyond 64), or one field split over a cluster of
    8 CTAs that transpose through distributed shared memory (ssp_cluster.cu: N = 128 at B <= 64);
    with planes the row / column kernels run.  Same transforms, same tables: the paths agree to fp32 rounding, and one
    launch replaces 2 n_steps + 1."""
    import torch
    n_steps, S = 6, 5
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, 200 + N)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    l0 = ssp.launch_count()
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), **kw)
    assert ssp.launch_count() - l0 == 1
    planes = torch.empty((B, n_steps, N, N), dtype=torch.complex64, device="cuda")
    out_mk = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), planes=planes, **kw)
    assert ssp.launch_count() - l0 == 1 + 2 * n_steps + 1
    assert rel_l2(out.cpu().numpy(), out_mk.cpu().numpy().astype(np.complex128)).max() < 1e-6
    ref = orc.propagate(N, dx, lam, dz, u0, scr, **kw)
    assert rel_l2(out.cpu().numpy(), ref).max() < tol(N, S)
    g = synth.random_field(N, B, 300 + N)
    gin = ssp.propagate_adjoint(N, dx, lam, list(dz), cu(g), cu(scr), **kw)
    gref = orc.propagate_adjoint(N, dx, lam, dz, g, scr, **kw)
    assert rel_l2(gin.cpu().numpy(), gref).max() < tol(N, S)


def test_odd_batch_and_vacuum_paths_at_1024(ssp, orc):
    """Edge cases of the TMA column kernel's persistent tile loop and of the fast / generic row instantiations:
    a batch that does not fill the last wave evenly (B = 3), vacuum only (S = 0), window off, one step."""
    N, dx, lam = 1024, 1e-3, 1e-6
    u0 = synth.random_field(N, 3, 77)
    scr = synth.random_screens(N, 3, 1, 78, rms=2.0)
    dz = np.array([N * dx * dx / lam * 0.2])
    for kw, s in ((dict(win_order=16, win_sigma_frac=0.47), scr), (dict(), scr), (dict(), None),
                  (dict(win_order=4, win_sigma_frac=0.4), None)):
        ref = orc.propagate(N, dx, lam, dz, u0, s, **kw)
        out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(s) if s is not None else None, **kw)
        assert rel_l2(out.cpu().numpy(), ref).max() < tol(N, 1), kw


@pytest.mark.parametrize("N", [1024, 2048])
def test_swapped_handover_common_vs_generic(ssp, N):
    """For N >= 1024 the TMA column kernel hands the field to the row kernel re/im-swapped (DESIGN.md section 6,
    packed pairs).  The common row instantiation assumes that form, the generic one (saved planes, phase gradient)
    reads a run-time flag: both must produce the same bits, forward and adjoint."""
    import torch
    B, n_steps, S = 2, 3, 3
    dx, lam, dz, u0, scr = _case(N, B, n_steps, S, 4000 + N)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    out = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), **kw)
    planes = torch.empty((B, n_steps, N, N), dtype=torch.complex64, device="cuda")
    out_g = ssp.propagate(N, dx, lam, list(dz), cu(u0), cu(scr), planes=planes, **kw)
    assert torch.equal(out, out_g)
    assert torch.equal(planes[:, -1], out)
    g = cu(synth.random_field(N, B, 4100 + N))
    gin = ssp.propagate_adjoint(N, dx, lam, list(dz), g, cu(scr), **kw)
    grad = torch.empty((B, S, N, N), dtype=torch.float32, device="cuda")
    gin_g = ssp.propagate_adjoint(N, dx, lam, list(dz), g, cu(scr), planes=planes, phase_grad=grad, **kw)
    assert torch.equal(gin, gin_g)
    assert torch.isfinite(grad).all()


@pytest.mark.parametrize("N", [128, 512, 1024, 2048, 4096])
def test_bitwise_determinism(ssp, N):
    """Race check by other means (compute-sanitizer is closed on this pool): the shared-memory exchanges, mbarrier /
    TMA pipelines and named barriers have no data race if repeated runs on the same inputs are bitwise identical.
    Fields, adjoint fields, evolved screens and the statistics records (per-block partials added in a fixed order, no
    atomics) are compared over five runs.  The tall grids run the column kernels whose thread groups share tile buffers
    (2048: two groups on three buffers; 4096: two column pairs taking turns on one exchange buffer): an odd batch gives
    the groups unequal tile counts."""
    import torch
    from paper_2604_07248_b200 import api
    B, S = (6, 3) if N <= 1024 else (3, 2)
    dx, lam, dz, u0, scr = _case(N, B, S, S, 400 + N)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    d_u0, d_scr = cu(u0), cu(scr)
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(N)
    noise = [torch.view_as_complex(torch.randn(B, S, N, N, 2, device="cuda", generator=gen)) for _ in range(2)]
    nsh = [torch.view_as_complex(torch.randn(B, S, 3, 3, 3, 2, device="cuda", generator=gen)) for _ in range(2)]
    first = None
    for run in range(5):
        st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        out = ssp.propagate(N, dx, lam, list(dz), d_u0, d_scr, stats=st, roi_frac=0.5, **kw)
        gin = ssp.propagate_adjoint(N, dx, lam, list(dz), out, d_scr, **kw)
        out_as = ssp.propagate(N, dx, lam, list(dz), d_u0, d_scr, h_kind=api.H_ANGULAR_SPECTRUM, **kw)
        spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
        shc = torch.zeros((B, S, 3, 3, 3), dtype=torch.complex64, device="cuda")
        ssp.make_screens(N, dx, psd, lam, [1e-14] * S, [100.0] * S, 3, noise[0], nsh[0], spectrum=spec, sh_coef=shc)
        ev = ssp.evolve_screens(N, dx, psd, lam, [1e-14] * S, [100.0] * S, 3, 0.99, 0.3, -0.2, 0.01, noise[1], nsh[1], spec, shc)
        got = [out.clone(), gin.clone(), out_as.clone(), ev.clone(), spec.clone(), st.clone()]
        if first is None:
            first = got
        else:
            for a, b in zip(got, first):
                assert torch.equal(a, b), run
