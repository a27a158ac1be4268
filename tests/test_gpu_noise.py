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
    for frame in (0, 1):
        ssp.frame_host(N, dx, psd, lam, cn2, dz, n_sh, 0.97, 3.0, -2.0, 1e-3, 77, frame, h_in, h_out, h_st, 0.5,
                       d_field, spec, shc, scr, d_noise, d_nsh, d_st, ws, **kw)
        ssp.fill_noise(77, 2 * frame, noise)
        if n_sh:
            ssp.fill_noise(77, 2 * frame + 1, nsh_c)
        scr_ref = ssp.evolve_screens(N, dx, psd, lam, cn2, dz, n_sh, 0.97, 3.0, -2.0, 1e-3, noise, nsh_c if n_sh else None,
                                     spec2, shc2 if n_sh else None)
        st_ref = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device=dev)
        out_ref = ssp.propagate(N, dx, lam, dz, u0.cuda(), scr_ref, stats=st_ref, roi_frac=0.5, **kw)
        assert torch.equal(scr, scr_ref) and torch.equal(spec, spec2)
        assert torch.equal(h_out, out_ref.cpu())
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
