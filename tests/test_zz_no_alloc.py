"""mlens_map_histogram_static against mlens_map_histogram.

Some users of this library may not let it allocate on the device: their own memory manager has taken the whole GPU
(a serving process, a framework's caching allocator at its cap), or they sit on a path where an allocation's stall or
failure cannot be tolerated.  For them the histogram has a second entry point whose only scratch, the bin-edge table,
is a fixed 32 KB array inside the library image.  Here it must give the same counts as the allocating entry point,
to the last unit (both decide every pixel by comparisons with the same float64 edges), on calls made back to back
that share the table -- the second with fewer bins than the first, so it runs over the first one's leftovers.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should hide no other test.
It needs nothing from the other tests (its map is made here, from a seed) and passes alone in a fresh process too.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ml():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2506_02114_b200 as ml
    ml.lib()
    return ml


def _synthetic_map(n, seed):
    """Magnification-like values: log-normal about mu = 2 over four decades, with the values a histogram has to put
    somewhere sensible mixed in (zeros, negatives, NaN, infinities, denormals)."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    m = 2.0 * torch.exp(1.5 * torch.randn(n, generator=g, device="cuda", dtype=torch.float64))
    odd = torch.tensor([0.0, -1.0, float("nan"), float("inf"), -float("inf"), 5e-324, 1e300, 2.0], dtype=torch.float64, device="cuda")
    m[:: n // 64][: odd.numel()] = odd
    return m


def test_static_histogram_matches_allocating_path(ml):
    import torch
    n = 3_000_017                                   # several waves of blocks, four-load rounds and a ragged tail
    m = _synthetic_map(n, 20250602)
    mu_ref = 2.0
    calls = [(ml.HIST_STATIC_MAXBINS, -2.0, 2.0), (50, -1.5, 1.5), (7, 0.3, 0.31), (1, -1.0, 1.0), (ml.HIST_STATIC_MAXBINS, -2.0, 2.0)]
    outs = [torch.full((nb + 2,), -7, dtype=torch.int64, device="cuda") for nb, _, _ in calls]   # garbage: must be overwritten
    # Calls in a row on one stream, no synchronisation in between: each must see its own edges, not its neighbour's.
    ml.histogram_static(m, mu_ref, *calls[0][1:], calls[0][0], outs[0])     # (also the one-time set-up on this device)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (nb, lo, hi), out in zip(calls[1:], outs[1:]):
        assert ml.histogram_static(m, mu_ref, lo, hi, nb, out) is out
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after == free_before, "the device's free memory moved across calls that must not allocate"
    for (nb, lo, hi), out in zip(calls, outs):
        want = ml.histogram(m, mu_ref, lo, hi, nb)                            # the existing, allocating path
        assert torch.equal(out, want), f"nbins={nb}"
        assert int(out.sum()) == n
    assert torch.equal(outs[0], outs[-1])
    # empty map: counts cleared, nothing launched on the data
    out = torch.full((12,), 3, dtype=torch.int64, device="cuda")
    ml.histogram_static(m[:0], mu_ref, -1.0, 1.0, 10, out)
    assert int(out.abs().sum()) == 0


def test_static_histogram_refuses_what_it_cannot_hold(ml):
    import torch
    m = _synthetic_map(4096, 1)
    nb = ml.HIST_STATIC_MAXBINS + 1
    with pytest.raises(ml.MlensError, match="MLENS_HIST_STATIC_MAXBINS"):
        ml.histogram_static(m, 2.0, -2.0, 2.0, nb, torch.zeros(nb + 2, dtype=torch.int64, device="cuda"))
    with pytest.raises(ml.MlensError):                                        # host arrays would need a staging buffer
        ml.histogram_static(m.cpu().numpy(), 2.0, -2.0, 2.0, 8, np.zeros(10, dtype=np.uint64))
    # a host pointer handed straight to the C entry point is refused there too, before any kernel sees it
    import ctypes as C
    host = np.ones(16)
    out = torch.zeros(10, dtype=torch.int64, device="cuda")
    rc = ml.lib().mlens_map_histogram_static(host.ctypes.data, C.c_int64(16), C.c_double(2.0), C.c_double(-1.0), C.c_double(1.0),
                                             C.c_int32(8), out.data_ptr(), None)
    assert rc == -1 and b"device memory" in ml.lib().mlens_last_error()
    with pytest.raises(ml.MlensError):
        ml.histogram_static(m, -1.0, 0.0, 1.0, 4, torch.zeros(6, dtype=torch.int64, device="cuda"))
