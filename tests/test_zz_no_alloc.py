"""hft_diagnostics_noalloc (include/hft.h): the flux diagnostics of a caller-held field with the CTA partial sums in the
library's static device array instead of the context's cudaMalloc'ed buffer -- checked against hft_diagnostics (the
existing path) on two calls in a row, the second on different data so that what the first call left in the shared array
would show.  Collected last on purpose (the run uses pytest -x)."""
import numpy as np
import pytest
import torch

from paper_2501_06377_b200 import workloads as wl

pytestmark = pytest.mark.gpu

# the two paths run the same kernels in the same summation order: equal to the last bit; the bound the diagnostics tests
# use for fp64 sums (relative to the unsigned flux) is kept as the stated tolerance
RTOL = 1e-13


def hft():
    from paper_2501_06377_b200 import hft as m
    return m


def full_field(ctx):
    return torch.stack([ctx.get_full(r) for r in range(ctx.n_real)]).contiguous()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_noalloc_diagnostics_match_existing_path_twice(dtype):
    H = hft()
    w = wl.scaled(wl.config(3), 61, 200, n_real=5)               # ragged: 200 columns, 61 rows over 64 partial-sum CTAs
    tdt = torch.float64 if dtype == "f64" else torch.float32
    ctx = H.Context(w.n_theta, w.n_phi, w.params, dtype=dtype)
    maps = wl.initial_maps(w).to(tdt)
    out = torch.full((w.n_real, 4), float("nan"), dtype=torch.float64, device="cuda")
    for call in range(2):
        for r in range(w.n_real):
            m = maps[r] if call == 0 else (-0.37 * (r + 1)) * maps[(r + 1) % w.n_real].flip(1) + 0.25
            ctx.set_map(r, m.contiguous().cuda())
        want = ctx.diagnostics()                                 # existing path: context buffer, host result
        field = full_field(ctx)                                  # the caller's copy [R][nt+2][np]
        before = torch.cuda.memory_allocated()
        ctx.diagnostics_noalloc(field, out)
        assert torch.cuda.memory_allocated() == before
        ctx.synchronize()
        got = out.cpu().numpy()
        scale = np.abs(want[:, 1:2])
        assert np.isfinite(got).all()
        assert (np.abs(got - want) <= RTOL * scale).all(), (call, got, want)
        assert np.array_equal(got, want)                         # same kernels, same order


def test_noalloc_rejects_more_realizations_than_the_static_array_holds():
    H = hft()
    n = 1025                                                     # HFT_NOALLOC_MAX_REAL = 1024
    params = np.tile(np.asarray(wl.config(3).params)[:1], (n, 1))
    ctx = H.Context(8, 32, params, dtype="f32")
    field = torch.zeros((n, 10, 32), dtype=torch.float32, device="cuda")
    out = torch.zeros((n, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(Exception) as ei:
        ctx.diagnostics_noalloc(field, out)
    assert "invalid argument" in str(ei.value) and "HFT_NOALLOC_MAX_REAL = 1024" in str(ei.value)   # hft_last_cuda_error text
