"""tb_series_mean_noalloc: the one entry point of libtb that allocates no device memory.

Why it exists: some users of the library cannot let it call cudaMalloc.  A telescope back end's real-time
loop cannot, because cudaMalloc / cudaFree serialise on the driver and make the device drain, which stalls
the ingest copies and searches running on its other streams; a process that gave all GPU memory to its own
pool at start-up cannot, because cudaMalloc then has nothing to return.  For them the fill value of a new
series (its fp64 mean, reading G8) is computed with the reduction's scratch in a static device array of
tb.TB_NOALLOC_SCRATCH_BYTES that is shared by every call in the process.

What is checked: on two calls in a row (no synchronisation between them, second series shorter than the
first, so stale partial sums of call 1 sit in the shared array during call 2) the result equals the fill
value of the existing, allocating path -- a plan created on the same series -- under the comparison the
fill-value tests of test_gpu_parity.py use (identical float32), and the fp64 mean itself to 1e-13 relative
(against a float64 numpy sum).  Lengths beyond the array's capacity are refused with a message that says so.

The file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.
It passes on its own in a fresh process and after the rest of the suite (the entry point does its one-off
address look-up on its first call, whenever that is).
"""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def tb():
    from paper_2112_11991_b200 import build
    build.build()
    from paper_2112_11991_b200 import tb
    return tb


def _mean_f64(x):
    return float(np.sum(np.asarray(x, dtype=np.float64)) / len(x))


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_plans_fill_value(tb, c1):
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(0)
    rng = np.random.default_rng(20211222)
    first = (rng.standard_normal(1 << 20) * 7.0 + 3.0).astype(np.float32)        # 16 tiles of 65 536
    second = np.ascontiguousarray(c1.series + np.float32(3.0), dtype=np.float32)  # 2 tiles; same series as
    assert len(second) < len(first)                                               # test_default_fill_is_the_series_mean

    # the caller's own buffers (here torch's; the entry point itself allocates nothing)
    d_first, d_second = torch.from_numpy(first).cuda(), torch.from_numpy(second).cuda()
    d_out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    torch.cuda.synchronize()
    tb.tb_series_mean_noalloc(d_first.data_ptr(), len(first), d_out.data_ptr(), stream)
    tb.tb_series_mean_noalloc(d_second.data_ptr(), len(second), d_out.data_ptr() + 8, stream)
    torch.cuda.synchronize()
    got = d_out.cpu().numpy()

    for series, mean in ((first, got[0]), (second, got[1])):
        with tb.Plan(series, c1.tsamp) as plan:                  # the existing path: cudaMalloc + k_sum_f64 + host sum
            fill = plan.info()["fill_value"]
        assert np.float32(mean) == np.float32(fill), (mean, fill)
        assert abs(mean - _mean_f64(series)) <= 1e-13 * max(1.0, abs(_mean_f64(series)))

    # the same two again, in the other order, plus a ragged length that ends inside a tile: the shared
    # array now holds sixteen stale tile sums and a counter that was used twice
    ragged = first[: 3 * 65536 + 12345]
    d_out.fill_(float("nan"))
    d_out3 = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    tb.tb_series_mean_noalloc(d_second.data_ptr(), len(second), d_out.data_ptr() + 8, stream)
    tb.tb_series_mean_noalloc(d_first.data_ptr(), len(ragged), d_out3.data_ptr(), stream)
    tb.tb_series_mean_noalloc(d_first.data_ptr(), len(first), d_out.data_ptr(), stream)
    torch.cuda.synchronize()
    again = d_out.cpu().numpy()
    assert again[0] == got[0] and again[1] == got[1], "the result must not depend on what the array held before"
    assert abs(float(d_out3.cpu()[0]) - _mean_f64(ragged)) <= 1e-13 * abs(_mean_f64(ragged))
    one = torch.tensor([-2.5], dtype=torch.float32, device="cuda")
    tb.tb_series_mean_noalloc(one.data_ptr(), 1, d_out3.data_ptr(), stream)
    torch.cuda.synchronize()
    assert float(d_out3.cpu()[0]) == -2.5


@pytest.mark.gpu
def test_host_pointers_are_refused(tb):
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    host = np.zeros(1024, dtype=np.float32)
    d_out = torch.zeros(1, dtype=torch.float64, device="cuda")
    with pytest.raises(tb.TbError) as ei:
        tb.tb_series_mean_noalloc(host.ctypes.data, len(host), d_out.data_ptr())
    assert ei.value.code == tb.TB_ERR_INVALID_ARG and "device memory" in str(ei.value)


def test_sizes_beyond_the_static_array_are_refused(tb):
    """Argument checks come before any CUDA call, so this part runs without a GPU: nothing is read or queued."""
    fake = 0x1000                                                # never dereferenced
    with pytest.raises(tb.TbError) as ei:
        tb.tb_series_mean_noalloc(fake, tb.TB_NOALLOC_MAX_SAMPLES + 1, fake)
    assert ei.value.code == tb.TB_ERR_CAPACITY
    assert "TB_NOALLOC_MAX_SAMPLES = 268435456" in str(ei.value) and "268435457" in str(ei.value)
    with pytest.raises(tb.TbError) as ei:
        tb.tb_series_mean_noalloc(fake, 0, fake)
    assert ei.value.code == tb.TB_ERR_INVALID_ARG
    with pytest.raises(tb.TbError) as ei:
        tb.tb_series_mean_noalloc(None, 16, fake)
    assert ei.value.code == tb.TB_ERR_INVALID_ARG
    assert tb.TB_NOALLOC_SCRATCH_BYTES == (32 + (tb.TB_NOALLOC_MAX_SAMPLES >> 16)) * 8
