"""ssp_fill_noise against the oracle's independent generator (Q29): the Philox words are integers, so a single
wrong bit shows as an O(1) difference; the floats agree to fp32 rounding of log / sqrt / sincospi."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ssp():
    from paper_2604_07248_b200 import api, build
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    ctx = api.Context(0)
    yield ctx
    ctx.close()


@pytest.mark.parametrize("seed,stream,first,n", [
    (1, 0, 0, 4096), (2604, 7248, 0, 100003),                 # odd count: ragged tail
    (0xDEADBEEF12345678, 0xABCDEF0123456789, 1 << 33, 70000), # high halves of seed / stream, block index beyond 2^32
    (7, 1, (1 << 33) - 1000, 3000),                           # straddles the 2^32 block boundary
    (5, 5, 0, 1), (5, 5, 0, 2)])
def test_fill_noise_matches_oracle(ssp, orc, seed, stream, first, n):
    out = torch.zeros(n + 8, dtype=torch.complex64, device="cuda")
    ssp.fill_noise(seed, stream, out[:n], first=first)
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.complex128)
    ref = orc.noise(seed, stream, n, first=first)
    # sin / cos from the special-function unit: absolute error ~2^-21 = 5e-7, times r <= 5.8, plus the rounding of
    # pi g (2e-7 in the angle) and of log / sqrt (1e-7 relative): |error| <= 1e-6 (1 + |z|), typically a few 1e-7
    err = np.abs(got[:n] - ref)
    assert np.all(err < 1e-6 * (1 + np.abs(ref))), (err.max(), err.argmax())
    assert np.sqrt(np.mean(err ** 2)) < 1e-6
    assert np.all(got[n:] == 0)                                # nothing written past the end


def test_fill_noise_feeds_the_screen_generator(ssp, orc):
    """A screen stack made from device-filled noise equals the oracle's screens made from the oracle's own draws."""
    from paper_2604_07248_b200 import api
    N, dx, lam, S, B, n_sh = 256, 2e-3, 1.55e-6, 2, 2, 2
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=20.0, l0=4e-3)
    noise = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    nsh = torch.empty((B, S, n_sh, 3, 3), dtype=torch.complex64, device="cuda")
    ssp.fill_noise(42, 0, noise)
    ssp.fill_noise(42, 1, nsh)
    scr = ssp.make_screens(N, dx, psd, lam, [1e-14] * S, [100.0] * S, n_sh, noise, nsh).cpu().numpy()
    pairs = lambda z, shape: np.stack([z.real, z.imag], axis=-1).astype(np.float32).reshape(*shape, 2)
    o_noise = pairs(orc.noise(42, 0, B * S * N * N), (B, S, N, N))
    o_nsh = pairs(orc.noise(42, 1, B * S * n_sh * 9), (B, S, n_sh, 3, 3))
    ref = orc.make_screens(N, dx, orc.Psd(kind=1, L0=20.0, l0=4e-3), lam, [1e-14] * S, [100.0] * S, n_sh, o_noise, o_nsh)[0]
    for b in range(B):
        for s in range(S):
            rel = np.linalg.norm(scr[b, s] - ref[b, s]) / np.linalg.norm(ref[b, s])
            assert rel < 2e-5 * np.log2(N), (b, s, rel)


@pytest.mark.parametrize("B,n_sh", [(1, 0), (11, 3), (16, 1)])
def test_frame_host_equals_the_separate_calls(ssp, B, n_sh):
    """ssp_frame_host (chunked, overlapped) returns bit for bit what fill_noise + evolve_screens + propagate return on
    the whole batch (those are each checked against the oracle), over two successive frames."""
    from paper_2604_07248_b200 import api, synth
    N, dx, lam, S = 128, 2e-3, 1.55e-6, 3
    cn2, dz = [1e-14, 3e-14, 2e-15], [100.0, 40.0, 250.0]
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=20.0, l0=4e-3)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    dev = "cuda"
    c64 = lambda *sh: torch.empty(sh, dtype=torch.complex64, device=dev)
    noise, nsh = c64(B, S, N, N), c64(B, S, max(n_sh, 1), 3, 3)
    ssp.fill_noise(9, 100, noise)
    spec, shc = c64(B, S, N, N), torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device=dev)
    nsh_c = nsh                                                  # [B][S][n_sh][3][3] when n_sh > 0
    if n_sh:
        ssp.fill_noise(9, 101, nsh_c)
    ssp.make_screens(N, dx, psd, lam, cn2, dz, n_sh, noise, nsh_c if n_sh else None, spectrum=spec, sh_coef=shc if n_sh else None)
    spec2, shc2 = spec.clone(), shc.clone()
    u0 = torch.from_numpy(synth.gaussian_beam(N, dx, 3e-2, B))
    h_in, h_out = u0.pin_memory(), torch.empty_like(u0).pin_memory()
    h_st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8).pin_memory()
    Bc = api.frame_chunk(B)
    d_field, scr = c64(B, N, N), torch.empty((B, S, N, N), dtype=torch.float32, device=dev)
    d_noise, d_nsh = c64(Bc, S, N, N), c64(B, S, max(n_sh, 1), 3, 3)
    d_st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device=dev)
    ws = ssp.workspace(N, dx, B, S)
    h_adj, d_adj = torch.empty_like(u0).pin_memory(), c64(B, N, N)
    for frame in (0, 1):
        adj = dict(h_adjoint_out=h_adj, d_adjoint=d_adj) if frame == 1 else {}      # frame 0: forward only
        ssp.frame_host(N, dx, psd, lam, cn2, dz, n_sh, 0.97, 3.0, -2.0, 1e-3, 77, frame, h_in, h_out, h_st, 0.5,
                       d_field, spec, shc, scr, d_noise, d_nsh, d_st, ws, **kw, **adj)
        ssp.fill_noise(77, 2 * frame, noise)
        if n_sh:
            ssp.fill_noise(77, 2 * frame + 1, nsh_c)
        scr_ref = ssp.evolve_screens(N, dx, psd, lam, cn2, dz, n_sh, 0.97, 3.0, -2.0, 1e-3, noise, nsh_c if n_sh else None,
                                     spec2, shc2 if n_sh else None)
        st_ref = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device=dev)
        out_ref = ssp.propagate(N, dx, lam, dz, u0.cuda(), scr_ref, stats=st_ref, roi_frac=0.5, **kw)
        assert torch.equal(scr, scr_ref) and torch.equal(spec, spec2)
        assert torch.equal(h_out, out_ref.cpu())
        if frame == 1:                                           # the adjoint leg: A^H of the received fields
            g_ref = ssp.propagate_adjoint(N, dx, lam, dz, out_ref, scr_ref, **kw)
            assert torch.equal(h_adj, g_ref.cpu())
        for a, b in zip(api.stats_to_dicts(h_st), api.stats_to_dicts(st_ref)):
            for k in ("power", "w2", "I_axis", "roi_sumI2"):
                assert abs(a[k] / b[k] - 1) < 1e-12


def test_fill_noise_errors(ssp):
    from paper_2604_07248_b200 import api
    out = torch.zeros(16, dtype=torch.complex64, device="cuda")
    with pytest.raises(api.SspError):
        ssp.fill_noise(1, 1, out, first=3)                     # odd first draw
    with pytest.raises(api.SspError):
        ssp.fill_noise(1, 1, out[1:])                          # 8-byte aligned only
    ssp.fill_noise(1, 1, out[:0])                              # empty: no-op


def test_philox_known_answer_vectors_on_device(ssp):
    """The device generator word for word against the published Philox-4x32-10 vectors (tests/golden/philox_kat.txt,
    Salmon et al. SC'11): counter (i lo, i hi, stream lo, stream hi), key (seed lo, seed hi) as DESIGN.md Q29 states."""
    from tests.test_oracle_noise import philox_kat_vectors
    for ctr, key, want in philox_kat_vectors():
        i = ctr[0] | (ctr[1] << 32)
        stream = ctr[2] | (ctr[3] << 32)
        seed = key[0] | (key[1] << 32)
        w = ssp.philox_words(seed, stream, i, 1).cpu().numpy().view(np.uint32)[0]
        assert [int(v) for v in w] == want, ([hex(int(v)) for v in w], [hex(v) for v in want])


def test_philox_words_are_what_fill_noise_draws_from(ssp, orc):
    """ssp_philox_words and ssp_fill_noise share one device function: Box-Muller (in fp64, here) on the words equals the draws,
    and the words equal the oracle's independent integer implementation bit for bit, ragged block counts included."""
    seed, stream, first_block, nb = 0x0123456789ABCDEF, 0xFEDCBA9876543210, (1 << 32) - 3, 1029
    w = ssp.philox_words(seed, stream, first_block, nb).cpu().numpy().view(np.uint32)
    idx = np.arange(first_block, first_block + nb, dtype=np.uint64)
    ctr = np.stack([idx & np.uint64(0xFFFFFFFF), idx >> np.uint64(32),
                    np.full(nb, stream & 0xFFFFFFFF, dtype=np.uint64), np.full(nb, stream >> 32, dtype=np.uint64)], axis=1)
    ref = orc.philox4x32_10(ctr.astype(np.uint32), (seed & 0xFFFFFFFF, seed >> 32))
    assert np.array_equal(w, ref)
    out = torch.zeros(2 * nb, dtype=torch.complex64, device="cuda")
    ssp.fill_noise(seed, stream, out, first=2 * first_block)
    x = w.astype(np.float64).reshape(-1, 2)
    u = (np.floor(x[:, 0] / 512.0) + 0.5) / 8388608.0
    f = (np.floor(x[:, 1] / 512.0) + 0.5) / 8388608.0
    z = np.sqrt(-2.0 * np.log(u)) * np.exp(2j * np.pi * f)
    assert np.all(np.abs(out.cpu().numpy() - z) < 1e-6 * (1 + np.abs(z)))


def test_frame_host_rejects_bad_arguments_before_any_copy(ssp):
    """A bad dz / a / S in ssp_frame_host is an SSP_EINVAL raised before anything is queued: the host output buffer is
    untouched, and the same buffers then serve a valid call whose result equals a fresh run."""
    from paper_2604_07248_b200 import api, synth
    N, dx, lam, S, B, n_sh = 128, 2e-3, 1.55e-6, 3, 4, 2
    cn2, dz = [1e-14, 3e-14, 2e-15], [100.0, 40.0, 250.0]
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=20.0, l0=4e-3)
    kw = dict(win_order=16, win_sigma_frac=0.47)
    c64 = lambda *sh: torch.empty(sh, dtype=torch.complex64, device="cuda")
    noise, nsh = c64(B, S, N, N), c64(B, S, n_sh, 3, 3)
    ssp.fill_noise(9, 100, noise)
    ssp.fill_noise(9, 101, nsh)
    spec, shc = c64(B, S, N, N), c64(B, S, n_sh, 3, 3)
    ssp.make_screens(N, dx, psd, lam, cn2, dz, n_sh, noise, nsh, spectrum=spec, sh_coef=shc)
    spec0, shc0 = spec.clone(), shc.clone()
    u0 = torch.from_numpy(synth.gaussian_beam(N, dx, 3e-2, B))
    h_in = u0.pin_memory()
    h_out = torch.full_like(u0, 7.0 + 7.0j).pin_memory()
    h_st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8).pin_memory()
    Bc = api.frame_chunk(B)
    d_field, scr = c64(B, N, N), torch.empty((B, S, N, N), dtype=torch.float32, device="cuda")
    d_noise, d_nsh = c64(Bc, S, N, N), c64(B, S, n_sh, 3, 3)
    d_st = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    ws = ssp.workspace(N, dx, B, S)
    d_field.zero_()
    run = lambda dz_, a_: ssp.frame_host(N, dx, psd, lam, cn2, dz_, n_sh, a_, 3.0, -2.0, 1e-3, 77, 0, h_in, h_out, h_st, 0.5,
                                         d_field, spec, shc, scr, d_noise, d_nsh, d_st, ws, **kw)
    for bad_dz, bad_a in (([100.0, -40.0, 250.0], 0.97), ([100.0, 40.0, float("nan")], 0.97), (dz, 1.5)):
        with pytest.raises(api.SspError) as ei:
            run(bad_dz, bad_a)
        assert ei.value.code == api.EINVAL
        torch.cuda.synchronize()
        assert torch.all(h_out == 7.0 + 7.0j)                  # nothing was copied back
        assert torch.all(d_field == 0)                         # nothing was uploaded
        assert torch.equal(spec, spec0) and torch.equal(shc, shc0)   # the AR state did not advance
    run(dz, 0.97)
    got = h_out.clone()
    spec.copy_(spec0); shc.copy_(shc0)
    run(dz, 0.97)
    assert torch.equal(got, h_out) and torch.all(torch.isfinite(torch.view_as_real(h_out)))


@pytest.mark.parametrize("N,kind,wind,n_sh,first", [
    (512, "vk", False, 3, 0), (512, "ocean", True, 2, 1 << 33), (1024, "vk", True, 3, 6 * 1024 * 1024), (1024, "ocean", False, 0, 2),
    (2048, "vk", True, 2, 4), (4096, "ocean", False, 1, 1 << 34)])       # the register-load generator of the tall grids
def test_seeded_evolution_equals_fill_noise_plus_evolve(ssp, orc, N, kind, wind, n_sh, first):
    """ssp_evolve_screens_seeded draws the fresh noise inside the generator's column kernel (Philox blocks shared by the
    two lanes that own adjacent columns): screens and the advanced spectrum must be the very bytes of ssp_fill_noise +
    ssp_evolve_screens, over two frames (the second starts from the first's spectrum), with and without wind, both PSD
    code paths, a draw offset past 2^32 blocks; at 512 the result is also checked against the oracle fed with the
    oracle's own draws."""
    from paper_2604_07248_b200 import api
    B, S, dx, lam = (2 if N <= 2048 else 1), 3, 2e-3, 1.0e-6
    psd_kw = dict(kind=api.PSD_VON_KARMAN, L0=10.0, l0=5e-3) if kind == "vk" else \
        dict(kind=api.PSD_OCEAN_NIKISHOV, eps=1e-5, chi_T=1e-7, w=-2.0, eta=1e-3)
    psd = api.PsdParams(**psd_kw)
    cn2, dz = [2e-14, 1e-14, 3e-14], [80.0, 120.0, 100.0]
    a, (vx, vy, T) = 0.97, ((0.8, -0.4, 5e-3) if wind else (0.0, 0.0, 0.0))
    seed = 2604 + N
    gen = torch.Generator(device="cuda").manual_seed(N + n_sh)
    noise0 = torch.view_as_complex(torch.randn(B, S, N, N, 2, device="cuda", generator=gen))
    nsh = [torch.view_as_complex(torch.randn(B, S, max(n_sh, 1), 3, 3, 2, device="cuda", generator=gen)) for _ in range(3)]
    state = []
    for _ in range(2):                                         # the same initial spectrum for both paths
        spec = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
        shc = torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device="cuda")
        ssp.make_screens(N, dx, psd, lam, cn2, dz, n_sh, noise0, nsh[0], spectrum=spec, sh_coef=shc)
        state.append((spec, shc))
    fresh = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    for frame in (1, 2):
        off = first + (frame - 1) * B * S * N * N
        ssp.fill_noise(seed, 2 * frame, fresh, first=off)
        ref = ssp.evolve_screens(N, dx, psd, lam, cn2, dz, n_sh, a, vx, vy, T, fresh, nsh[frame], state[0][0], state[0][1])
        got = ssp.evolve_screens_seeded(N, dx, psd, lam, cn2, dz, n_sh, a, vx, vy, T, seed, 2 * frame, off, nsh[frame],
                                        state[1][0], state[1][1])
        assert torch.equal(got, ref), (frame, float((got - ref).abs().max()))
        assert torch.equal(state[1][0], state[0][0]) and torch.equal(state[1][1], state[0][1]), frame
    if N == 512:
        # against the oracle: its own generator for the draws, its own evolution (one frame from a zero spectrum)
        spec = torch.zeros((B, S, N, N), dtype=torch.complex64, device="cuda")
        shc = torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device="cuda")
        got = ssp.evolve_screens_seeded(N, dx, psd, lam, cn2, dz, n_sh, 0.0, vx, vy, T, seed, 7, first, nsh[0], spec, shc)
        hi = orc.noise(seed, 7, B * S * N * N, first=first).reshape(B, S, N, N)
        sh = nsh[0].cpu().numpy().astype(np.complex128)[:, :, :n_sh]
        ref, _, _ = orc.make_screens(N, dx, orc.Psd(**{k: v for k, v in psd_kw.items()}), lam, cn2, dz, n_sh,
                                     np.stack([hi.real, hi.imag], -1), np.stack([sh.real, sh.imag], -1), keep_spectrum=False)
        err = np.sqrt(np.sum((got.cpu().numpy() - ref) ** 2, axis=(-2, -1)) / np.sum(ref ** 2, axis=(-2, -1)))
        assert err.max() < 2e-5 * np.log2(N), err.max()


def test_seeded_evolution_rejects_small_grids_and_odd_offsets(ssp):
    from paper_2604_07248_b200 import api
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    for N in (64, 256):
        spec = torch.zeros((1, 1, N, N), dtype=torch.complex64, device="cuda")
        shc = torch.zeros((1, 1, 1, 3, 3), dtype=torch.complex64, device="cuda")
        with pytest.raises(api.SspError) as e:
            ssp.evolve_screens_seeded(N, 1e-3, psd, 1e-6, [1e-14], [100.0], 0, 0.9, 0, 0, 0, 1, 2, 0, None, spec, shc)
        assert e.value.code == api.EUNSUPPORTED
    spec = torch.zeros((1, 1, 512, 512), dtype=torch.complex64, device="cuda")
    with pytest.raises(api.SspError) as e:                     # odd first draw
        ssp.evolve_screens_seeded(512, 1e-3, psd, 1e-6, [1e-14], [100.0], 0, 0.9, 0, 0, 0, 1, 2, 3, None, spec, None)
    assert e.value.code == api.EINVAL


def test_seeded_evolution_across_generator_chunks(ssp):
    """The generator works through B x S screens in chunks of 512 MB of column-transformed spectra (256 screens at 512^2);
    the seeded kernel's draw index must continue across the chunk boundary: 300 screens, one frame, bytes of fill + evolve."""
    from paper_2604_07248_b200 import api
    N, B, S, dx, lam, n_sh = 512, 30, 10, 2e-3, 1.0e-6, 1
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=10.0, l0=5e-3)
    cn2, dz = [1e-14] * S, [100.0] * S
    gen = torch.Generator(device="cuda").manual_seed(5)
    nsh = torch.view_as_complex(torch.randn(B, S, n_sh, 3, 3, 2, device="cuda", generator=gen))
    fresh = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    ssp.fill_noise(11, 4, fresh, first=2 * N * N)
    out = []
    for seeded in (False, True):
        spec = torch.zeros((B, S, N, N), dtype=torch.complex64, device="cuda")
        shc = torch.zeros((B, S, n_sh, 3, 3), dtype=torch.complex64, device="cuda")
        if seeded:
            scr = ssp.evolve_screens_seeded(N, dx, psd, lam, cn2, dz, n_sh, 0.5, 0.3, 0.1, 1e-2, 11, 4, 2 * N * N, nsh, spec, shc)
        else:
            scr = ssp.evolve_screens(N, dx, psd, lam, cn2, dz, n_sh, 0.5, 0.3, 0.1, 1e-2, fresh, nsh, spec, shc)
        out.append((scr, spec))
    assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1])
    assert float(out[1][0][-1].abs().max()) > 0                # the last chunk was written


@pytest.mark.parametrize("N,kind,n_sh,keep", [(512, "vk", 3, True), (1024, "ocean", 2, False), (1024, "vk", 0, True), (2048, "vk", 1, True)])
def test_seeded_first_synthesis_equals_fill_noise_plus_make(ssp, N, kind, n_sh, keep):
    """ssp_make_screens_seeded (no noise array at all) against ssp_fill_noise + ssp_make_screens: screens, and the stored
    spectrum / coefficients when kept, are the same bytes; a seeded evolution on top continues identically."""
    from paper_2604_07248_b200 import api
    B, S, dx, lam = 2, 2, 2e-3, 1.0e-6
    psd = api.PsdParams(kind=api.PSD_VON_KARMAN, L0=10.0, l0=5e-3) if kind == "vk" else \
        api.PsdParams(kind=api.PSD_OCEAN_NIKISHOV, eps=1e-5, chi_T=1e-7, w=-2.0, eta=1e-3)
    cn2, dz = [2e-14, 1e-14], [80.0, 120.0]
    gen = torch.Generator(device="cuda").manual_seed(N)
    nsh = torch.view_as_complex(torch.randn(B, S, max(n_sh, 1), 3, 3, 2, device="cuda", generator=gen))
    noise = torch.empty((B, S, N, N), dtype=torch.complex64, device="cuda")
    ssp.fill_noise(77, 0, noise, first=4 * N)
    mk = lambda: (torch.zeros((B, S, N, N), dtype=torch.complex64, device="cuda") if keep else None,
                  torch.zeros((B, S, max(n_sh, 1), 3, 3), dtype=torch.complex64, device="cuda") if keep else None)
    spec_a, shc_a = mk()
    spec_b, shc_b = mk()
    ref = ssp.make_screens(N, dx, psd, lam, cn2, dz, n_sh, noise, nsh, spectrum=spec_a, sh_coef=shc_a)
    got = ssp.make_screens_seeded(N, dx, psd, lam, cn2, dz, n_sh, 77, 0, 4 * N, B, noise_sh=nsh, spectrum=spec_b, sh_coef=shc_b)
    assert torch.equal(got, ref)
    if keep:
        assert torch.equal(spec_a, spec_b) and torch.equal(shc_a, shc_b)
        ssp.fill_noise(77, 2, noise)
        ref = ssp.evolve_screens(N, dx, psd, lam, cn2, dz, n_sh, 0.9, 0.2, 0.1, 1e-2, noise, nsh, spec_a, shc_a)
        got = ssp.evolve_screens_seeded(N, dx, psd, lam, cn2, dz, n_sh, 0.9, 0.2, 0.1, 1e-2, 77, 2, 0, nsh, spec_b, shc_b)
        assert torch.equal(got, ref) and torch.equal(spec_a, spec_b)
