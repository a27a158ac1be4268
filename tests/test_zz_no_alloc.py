"""GPU: ssp_beam_stats_static -- the beam statistics without any allocation (scratch in a library-resident device
array, include/ssp.h) -- against the existing ssp_beam_stats path.  Collected last on purpose (file name): the
run uses pytest -x.  Passes alone in a fresh process and after the other GPU tests: it makes its own context
and depends on no earlier call (the ticket counters of the shared array are cleared by every call)."""
import numpy as np
import pytest

from paper_2604_07248_b200 import synth

pytestmark = pytest.mark.gpu

KEYS = ("power", "w2", "sxx", "syy", "sxy", "I_axis", "roi_sumI", "roi_sumI2")


@pytest.fixture(scope="module")
def ssp():
    import torch
    from paper_2604_07248_b200 import api, build
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    ctx = api.Context(0)
    yield ctx
    ctx.close()


def _fields(N, B, seed):
    import torch
    dx = 1e-3
    u = (synth.random_field(N, B, seed) + 2.0 * synth.gaussian_beam(N, dx, 0.2 * N * dx, B)).astype(np.complex64)
    return dx, torch.from_numpy(np.ascontiguousarray(u)).cuda()


def _same(api, got, ref, dx, N, what):
    """The tolerance of the statistics tests in test_gpu_propagate.py (1e-6 relative, centroids 1e-7 of the grid)."""
    for a, r in zip(api.stats_to_dicts(got), api.stats_to_dicts(ref)):
        for k in KEYS:
            assert abs(a[k] - r[k]) <= 1e-6 * abs(r[k]), (what, k, a[k], r[k])
        assert abs(a["cx"] - r["cx"]) < 1e-7 * dx * N and abs(a["cy"] - r["cy"]) < 1e-7 * dx * N, what
        assert a["roi_n"] == r["roi_n"], what


def test_static_scratch_statistics_match_the_allocating_path_on_calls_in_a_row(ssp):
    import torch
    from paper_2604_07248_b200 import api
    # calls in a row on the one shared array, shapes chosen so that a later call reads fewer and differently placed
    # records than the one before left there: many blocks per field, one block per field, a batch at the limit, again
    cases = [(1024, 3, 0.25), (64, 300, 0.5), (256, 5, 1.0), (8, api.STATS_STATIC_MAX_FIELDS, 0.0), (1024, 3, 0.25),
             (2048, 1, 0.5)]
    data = [(N, roi) + _fields(N, B, 900 + i) for i, (N, B, roi) in enumerate(cases)]
    refs = [ssp.beam_stats(N, dx, u, roi_frac=roi)[0] for N, roi, dx, u in data]           # existing path
    outs = [torch.full((u.shape[0] * api.STATS_BYTES,), 0xA5, dtype=torch.uint8, device="cuda") for _, _, _, u in data]
    N, roi, dx, u = data[0]
    ssp.beam_stats_static(N, dx, u, outs[0], roi_frac=roi)                                   # first use loads the kernel
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    n0 = ssp.launch_count()
    for (N, roi, dx, u), out in zip(data, outs):                                             # back to back, no sync between
        ssp.beam_stats_static(N, dx, u, out, roi_frac=roi)
    torch.cuda.synchronize()
    assert ssp.launch_count() - n0 == len(data)                                              # one kernel per call
    assert torch.cuda.mem_get_info()[0] == free0, "the no-allocation entry point changed the free device memory"
    for (N, roi, dx, u), out, ref in zip(data, outs, refs):
        _same(api, out, ref, dx, N, (N, u.shape[0], roi))
        assert torch.equal(out, ref), "same sums in the same order: the records are the same bytes"


def test_static_scratch_rejects_what_does_not_fit(ssp):
    import torch
    from paper_2604_07248_b200 import api
    N, B = 8, api.STATS_STATIC_MAX_FIELDS + 1
    dx, u = _fields(N, B, 77)
    out = torch.zeros(B * api.STATS_BYTES, dtype=torch.uint8, device="cuda")
    with pytest.raises(api.SspError) as e:
        ssp.beam_stats_static(N, dx, u, out)
    assert e.value.code == api.EINVAL and "exceeds the static scratch" in str(e.value)
    with pytest.raises(api.SspError):
        ssp.beam_stats_static(N, dx, u[:2], None)                                            # d_stats is required
    assert not out.any()                                                                     # nothing was launched
    # the context is still usable, and so is the array
    ref, _ = ssp.beam_stats(N, dx, u[:4])
    got = ssp.beam_stats_static(N, dx, u[:4], out[:4 * api.STATS_BYTES])
    _same(api, got, ref, dx, N, "after the rejected calls")
