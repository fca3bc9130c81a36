"""bt_moments_static: the beam statistics for callers that may not allocate device memory.

Some programs that embed this library cannot let it call cudaMalloc: the application's own arena has taken all of HBM
already (a library allocation then fails or steals from it), or the step loop keeps several streams in flight and an
allocation would stall them all (cudaMalloc synchronises the device), or an allocation checker flags every device
allocation a library makes.  bt_moments_static serves them: the caller passes its six coordinate arrays and a 42-double
output, and the per-block partial sums go into one fixed array that lives inside libbt.so (432 KiB per GPU, at most
bt.MOMENTS_STATIC_MAX_PARTICLES particles per call, one call at a time per GPU).

What is checked: its result against the existing, allocating path (bt_beam_moments_device) on the same device arrays, with
the tolerance of tests/test_gpu_moments_parity.py (the two paths associate the fp64 sums differently, so they agree to
rounding, not bitwise), on calls made back to back -- the array is shared and keeps the previous call's rows, so a later call
with fewer rows, more rows, or other data must not see them -- and that a bunch beyond the limit is refused with a clear
message before anything is launched.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process (first call on the device = the address look-up) and after the
others (the other statistics tests have then used the allocating path on the same device)."""
import numpy as np
import pytest

import paper_2208_02382_b200 as bt
import workloads as W

pytestmark = pytest.mark.gpu


def _agree(got, ref):
    """|mean - ref| <= 1e-12 sigma + 4 eps |ref| and |cov - ref| <= 1e-12 sqrt(ref_ii ref_jj): test_gpu_moments_parity's bar."""
    mean, cov = got[:6], got[6:].reshape(6, 6)
    rm, rc = ref[:6], ref[6:].reshape(6, 6)
    sig = np.sqrt(np.diag(rc))
    assert np.all(np.abs(mean - rm) <= 1e-12 * sig + 4 * np.finfo(float).eps * np.abs(rm)), (mean - rm, sig)
    scale = np.outer(sig, sig)
    if np.all(scale > 0):
        assert np.max(np.abs(cov - rc) / scale) <= 1e-12, np.max(np.abs(cov - rc) / scale)
    else:
        assert np.max(np.abs(cov - rc)) <= 1e-12 * max(np.max(scale), 1e-300)
    assert np.array_equal(cov, cov.T)


def _both_paths(c, offset=0):
    """The bunch `c` in six CUDA tensors (shifted by `offset` doubles from their allocation, 1 = only 8-byte aligned):
    (result of bt_moments_static, result of bt_beam_moments_device), each 42 doubles."""
    import torch
    n = c[0].shape[0]
    backing = [torch.empty(n + offset, dtype=torch.float64, device="cuda") for _ in range(6)]
    tensors = [b[offset:] for b in backing]
    beam = bt.Beam(n, storage=tensors)          # the existing path needs a beam; it borrows the same arrays
    try:
        beam.upload(c)
        ref = torch.full((42,), float("nan"), dtype=torch.float64, device="cuda")
        beam.moments_device(ref)
        out = torch.full((42,), float("nan"), dtype=torch.float64, device="cuda")
        bt.moments_static([t.data_ptr() for t in tensors], n, out.data_ptr(), stream=beam.stream)
        beam.sync()
        return out.cpu().numpy(), ref.cpu().numpy()
    finally:
        beam.close()


def test_static_scratch_matches_the_allocating_path_on_calls_in_a_row():
    # rows used per call: 31, then 4 (27 stale rows behind them), then 1, then 31 again with other data and 8-byte alignment
    first = None
    for k, (n, cfg_id, offset) in enumerate([(1_000_001, 0, 0), (100_003, 2, 0), (4097, 0, 0), (1_000_000, 2, 1)]):
        c = W.make_bunch(W.config(cfg_id, n=n))
        if k == 1:
            c[0] += 1.0      # an offset, correlated bunch: the provisional centre matters
            c[1] += 0.7 * c[0]
        got, ref = _both_paths(c, offset)
        assert np.all(np.isfinite(got))
        _agree(got, ref)
        if k == 0:
            first = (c, got)
    # the same data again after the array has been used by other bunches: bit-identical (deterministic, nothing stale read)
    again, _ = _both_paths(first[0])
    assert np.array_equal(again, first[1])


def test_static_scratch_two_calls_back_to_back_on_one_stream_without_a_sync_between():
    """Two bunches of different sizes reduced one after the other on one stream, results read only at the end: the second
    launch reuses the rows and the counter the first one left."""
    import torch
    ca, cb = W.make_bunch(W.config(0, n=300_001)), W.make_bunch(W.config(2, n=70_001))
    ta = [torch.from_numpy(a).cuda() for a in ca]
    tb = [torch.from_numpy(a).cuda() for a in cb]
    outs = torch.full((2, 42), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    bt.moments_static([t.data_ptr() for t in ta], 300_001, outs[0].data_ptr(), stream=stream)
    bt.moments_static([t.data_ptr() for t in tb], 70_001, outs[1].data_ptr(), stream=stream)
    torch.cuda.synchronize()
    got = outs.cpu().numpy()
    for c, g in zip((ca, cb), got):
        _, ref = _both_paths(c)
        _agree(g, ref)


def test_static_scratch_refuses_what_does_not_fit():
    import torch
    t = [torch.zeros(16, dtype=torch.float64, device="cuda") for _ in range(6)]
    out = torch.zeros(42, dtype=torch.float64, device="cuda")
    before = bt.launch_count()
    with pytest.raises(bt.BtError) as ei:       # the size is checked before any pointer is touched
        bt.moments_static([x.data_ptr() for x in t], bt.MOMENTS_STATIC_MAX_PARTICLES + 1, out.data_ptr())
    assert ei.value.code == bt.BT_ERR_INVALID
    assert "BT_MOMENTS_STATIC_MAX_PARTICLES" in str(ei.value) and "bt_beam_moments_device" in str(ei.value)
    with pytest.raises(bt.BtError):
        bt.moments_static([x.data_ptr() for x in t], 0, out.data_ptr())
    with pytest.raises(bt.BtError):
        bt.moments_static([x.data_ptr() for x in t[:5]] + [0], 16, out.data_ptr())
    assert bt.launch_count() == before
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0


def test_static_scratch_at_the_limit():
    """n = BT_MOMENTS_STATIC_MAX_PARTICLES exactly: all 2048 rows in use (6 x 512 MiB of coordinates)."""
    import torch
    n = bt.MOMENTS_STATIC_MAX_PARTICLES
    g = torch.Generator(device="cuda").manual_seed(20220802)
    tensors = [torch.randn(n, dtype=torch.float64, device="cuda", generator=g) * (1e-3 * (i + 1)) + 0.01 * i for i in range(6)]
    beam = bt.Beam(n, storage=tensors)
    try:
        ref = torch.empty(42, dtype=torch.float64, device="cuda")
        beam.moments_device(ref)
        out = torch.empty(42, dtype=torch.float64, device="cuda")
        bt.moments_static([t.data_ptr() for t in tensors], n, out.data_ptr(), stream=beam.stream)
        beam.sync()
        _agree(out.cpu().numpy(), ref.cpu().numpy())
    finally:
        beam.close()
