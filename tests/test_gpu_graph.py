"""GPU: ssp_propagate / ssp_propagate_adjoint / ssp_beam_stats_static under CUDA graph capture.  After one call outside
capture (tables, TMA descriptors and the on-chip step list are cached by then) these calls issue kernels only -- no
allocation, no host copy -- so a frame can be captured once and replayed; the replay must produce the bytes of the eager
calls, also after the input buffers' contents have changed."""
import numpy as np
import pytest
import torch

from paper_2604_07248_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N,B", [(64, 3), (128, 4), (256, 8), (1024, 3)])
def test_captured_frame_replays_the_eager_result(N, B):
    from paper_2604_07248_b200 import api, build
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    S, dx, lam = 4, 1e-3, 1.0e-6
    dz = [N * dx * dx / lam * 0.2] * S
    kw = dict(win_order=16, win_sigma_frac=0.47)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        ctx = api.Context(0, stream=side)
        gen = torch.Generator(device="cuda").manual_seed(N)
        u0 = torch.from_numpy(synth.gaussian_beam(N, dx, 0.1 * N * dx, B)).cuda()
        scr = torch.randn(B, S, N, N, device="cuda", generator=gen)
        out, gin = torch.empty_like(u0), torch.empty_like(u0)
        stats = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
        stats2 = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")

        def frame():
            ctx.propagate(N, dx, lam, dz, u0, scr, out=out, stats=stats, **kw)
            ctx.propagate_adjoint(N, dx, lam, dz, out, scr, out=gin, **kw)
            ctx.beam_stats_static(N, dx, gin, stats2)

        frame()                                                # outside capture: everything cached
        side.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            frame()
        for trial in range(2):                                 # new contents in the same buffers
            u0.copy_(torch.view_as_complex(torch.randn(B, N, N, 2, device="cuda", generator=gen)))
            scr.copy_(torch.randn(B, S, N, N, device="cuda", generator=gen))
            frame()
            side.synchronize()
            want = [t.clone() for t in (out, gin, stats, stats2)]
            for t in (out, gin, stats, stats2):
                t.zero_()
            graph.replay()
            side.synchronize()
            for got, ref in zip((out, gin, stats, stats2), want):
                assert torch.equal(got, ref), (N, trial)
        del graph
        ctx.close()
