"""helios_rt_phase_curve_noalloc -- the phase curve for callers that cannot allocate device memory.

Some users of this library run where a cudaMalloc is not an option: a plug-in or host callback inside an application
that owns all of the GPU's memory and hands none out, a latency-critical path that must stay out of the driver's
allocator (an allocation can block, fail on a full device, or stall other streams), a worker whose memory budget is
already spent.  For them the library carries the phase curve's scratch itself, as a fixed 8 MiB device array, and
`phase_curve_noalloc` takes inputs and outputs only.

What is checked here, on a B200, through the C ABI:
  * its outputs equal those of the existing `phase_curve` (caller-allocated workspace) -- the two run the same
    kernels, so equal bit for bit, which is inside the 1e-12 tolerance the phase-curve parity test uses;
  * on two calls in a row, the second one smaller than the first and with other data: the built-in array is shared by
    all calls and still holds the first call's partial sums, and none of them may leak into the second result;
  * a problem that needs more than the 8 MiB is refused with the documented error code and leaves the output alone.

This file sorts last on purpose (pytest -x stops at the first failure; nothing may hide behind this test), and it
does not depend on what ran before it: it passes alone in a fresh process -- where its first call is the one that
looks up the array's address on the device -- and after the rest of the suite.
"""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    return torch


@pytest.fixture(scope="module")
def H():
    from paper_2203_02293_b200 import build, helios_rt
    build.build()
    return helios_rt


def _case(torch, level, nb, nph, seed):
    """Seeded phase-curve inputs on the icosahedral grid of the given refinement level, as CUDA tensors."""
    from paper_2203_02293_b200 import workloads as W
    lon, lat, area = W.grid_geometry(level)
    rng = np.random.default_rng(seed)
    F = 10 ** rng.uniform(-2, 4, (lon.size, nb))
    alpha = rng.uniform(-np.pi, np.pi, nph)
    edges = W.bin_edges_equal_wavenumber(nb)
    t = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda:0")
    return dict(F=t(F), lon=t(lon), lat=t(lat), area=t(area), alpha=t(alpha), edges=t(edges))


def _run(torch, fn, d, **kw):
    nph, nb = d["alpha"].shape[0], d["F"].shape[1]
    out = torch.full((nph, nb), float("nan"), dtype=torch.float64, device="cuda:0")
    band = torch.full((nph,), float("nan"), dtype=torch.float64, device="cuda:0")
    fn(d["F"], d["lon"], d["lat"], d["area"], d["alpha"], out, bin_edges=d["edges"], lam1=1.1e-6, lam2=1.7e-6,
       F_phase_band=band, **kw)
    return out, band


def test_noalloc_phase_curve_equals_the_workspace_path_on_two_calls_in_a_row(torch_cuda, H):
    torch = torch_cuda
    torch.cuda.set_device(0)
    # first call: 2562 columns (21 chunks, ragged tail), 301 bins (3 bin tiles, ragged), 37 phases (2 phase tiles):
    # 1.9 MB of the built-in array; second call: 642 columns, 30 bins, 5 phases -- a corner of what the first left.
    cases = [_case(torch, 4, 301, 37, seed=21), _case(torch, 3, 30, 5, seed=22)]
    expected = [_run(torch, H.phase_curve, d) for d in cases]      # existing path, workspace allocated by the binding
    torch.cuda.synchronize()
    got = [_run(torch, H.phase_curve_noalloc, d) for d in cases]   # two calls in a row, stream-ordered
    torch.cuda.synchronize()
    for (ref, ref_band), (out, band) in zip(expected, got):
        r, o = ref.cpu().numpy(), out.cpu().numpy()
        assert np.all(np.isfinite(o)) and np.all(np.isfinite(band.cpu().numpy()))
        # the tolerance of test_phase_curve_matches_the_oracle ...
        assert np.all(np.abs(o - r) <= 1e-12 * np.abs(r).max(axis=0, keepdims=True) + 1e-13 * np.abs(r))
        assert np.allclose(band.cpu().numpy(), ref_band.cpu().numpy(), rtol=1e-12, atol=0.0)
        # ... and, since both paths run the same kernels in the same order, in fact bit for bit
        assert torch.equal(out, ref) and torch.equal(band, ref_band)
    # and once more the large case, after the small one
    out, band = _run(torch, H.phase_curve_noalloc, cases[0])
    torch.cuda.synchronize()
    assert torch.equal(out, expected[0][0]) and torch.equal(band, expected[0][1])


def test_noalloc_phase_curve_refuses_what_does_not_fit(torch_cuda, H):
    torch = torch_cuda
    torch.cuda.set_device(0)
    lib = H.load_library()
    # the largest shape that fits and the first that does not (2562 columns = 21 chunks of 128, 64 phases)
    assert lib.helios_rt_phase_curve_workspace_bytes(2562, 780, 64) <= H.PHASE_CURVE_NOALLOC_MAX_BYTES
    assert lib.helios_rt_phase_curve_workspace_bytes(2562, 781, 64) > H.PHASE_CURVE_NOALLOC_MAX_BYTES
    d = _case(torch, 4, 781, 64, seed=23)
    out = torch.full((64, 781), -7.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(H.HeliosRTError, match=r"error -5: .*too large"):
        H.phase_curve_noalloc(d["F"], d["lon"], d["lat"], d["area"], d["alpha"], out)
    torch.cuda.synchronize()
    assert bool((out == -7.0).all())                   # refused before anything was queued
    # one bin fewer fits, runs, and matches the workspace path
    d = {k: (v[:, :780].contiguous() if k == "F" else v[:781] if k == "edges" else v) for k, v in d.items()}
    ref, ref_band = _run(torch, H.phase_curve, d)
    got, got_band = _run(torch, H.phase_curve_noalloc, d)
    torch.cuda.synchronize()
    assert torch.equal(got, ref) and torch.equal(got_band, ref_band)
