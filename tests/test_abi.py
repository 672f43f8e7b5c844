"""-m "not gpu": the C-ABI library loads and exports every symbol include/tb.h declares; host-only
entry points work; GPU entry points fail loudly (no CPU fallback) when there is no device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tb():
    from paper_2112_11991_b200 import build
    build.build()
    from paper_2112_11991_b200 import tb
    return tb


def test_every_declared_symbol_is_exported(tb):
    header = open(os.path.join(ROOT, "include", "tb.h")).read()
    declared = set(re.findall(r"\b(tb_[a-z0-9_]+)\s*\(", header))
    assert declared, "no declarations found"
    assert declared == set(tb.EXPORTS)
    for name in declared:
        assert hasattr(tb.lib, name), f"{name} not exported by libtb.so"


def test_struct_layouts_match_header(tb):
    assert ctypes.sizeof(tb.PlanOpts) == 88                      # + whiten, n_zap_ranges, zap_ranges, delay_model
    assert ctypes.sizeof(tb.Timings) == 6 * 8 + 7 * 8 + 2 * 8      # + ms_delay, fft_path_used
    assert tb.TEMPLATE_DTYPE.itemsize == 40 and tb.CANDIDATE_DTYPE.itemsize == 24
    assert ctypes.sizeof(tb.BankSpace) == 80                     # tb_bank_space


def test_host_only_entry_points(tb):
    from oracle import tb_oracle as orc
    for L in range(5):
        assert abs(tb.tb_sigma_to_power(L, 6.0) - orc.sigma_to_power(L, 6.0)) < 1e-9
    # survey table of 6-sigma power thresholds
    expect = [13.4376, 17.8476, 23.8993, 33.1819, 48.3992]
    for L, e in enumerate(expect):
        assert abs(tb.tb_sigma_to_power(L, 6.0) - e) < 5e-4
    with pytest.raises(tb.TbError):
        tb.tb_sigma_to_power(5, 6.0)
    assert tb.lib.tb_strerror(tb.TB_ERR_OVERFLOW) == b"candidate buffer overflow"
    assert tb.lib.tb_plan_destroy(None) == 0


def test_invalid_arguments_are_rejected_before_touching_the_gpu(tb):
    x = np.zeros(4096, dtype=np.float32)
    for n, tsamp, kw in [(4095, 1e-3, {}), (4096, 0.0, {}), (4096, -1.0, {}), (1024, 1e-3, {}),
                         (4096, 1e-3, {"median_window": 100}), (4096, 1e-3, {"median_window": 4096})]:
        with pytest.raises(tb.TbError) as ei:
            tb.tb_plan_create(x, n, tsamp, **kw)
        assert ei.value.code == tb.TB_ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_device(tb):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(tb.TbError) as ei:
        tb.tb_plan_create(np.zeros(4096, dtype=np.float32), 4096, 1e-3)
    assert ei.value.code == tb.TB_ERR_CUDA


def test_bank_host_entry_points_and_no_fallback(tb):
    """tb_bank_n_templates is host arithmetic (eq 18, 20, 21); the device entry points validate their
    arguments first and then fail with TB_ERR_CUDA when there is no GPU (no CPU path)."""
    import math
    import torch
    from oracle import tb_bank as obank
    for n_dim, vol in [(3, 1130.0), (5, 2.0e6)]:
        for exact in (True, False):
            assert tb.tb_bank_n_templates(0.9, 0.2, n_dim, vol, exact) == pytest.approx(obank.n_templates(0.9, 0.2, n_dim, vol, exact), rel=1e-12)
    assert tb.tb_bank_n_templates(0.9, 0.2, 3, 1e6, False) == pytest.approx(math.log(10) * 1e6 / (0.2 ** 1.5 * 4 * math.pi / 3))
    for bad in [(1.0, 0.2, 3, 10.0), (0.9, 0.0, 3, 10.0), (0.9, 0.2, 0, 10.0), (0.9, 0.2, 3, -1.0)]:
        with pytest.raises(tb.TbError):
            tb.tb_bank_n_templates(*bad)
    sp = tb.bank_space(537.0, 25.0, 53.7, 188.0)
    with pytest.raises(tb.TbError) as ei:
        tb.tb_bank_generate(tb.bank_space(-1.0, 25.0, 53.7, 188.0), np.zeros((4, 6)), 1.0)
    assert ei.value.code == tb.TB_ERR_INVALID_ARG
    if not torch.cuda.is_available():
        with pytest.raises(tb.TbError) as ei:
            tb.tb_bank_generate(sp, np.full((4, 6), 0.5), 1.0)
        assert ei.value.code == tb.TB_ERR_CUDA
        with pytest.raises(tb.TbError) as ei:
            tb.tb_bank_density(sp, np.array([[1.0, 0.05, 0.0, 0.0, 0.0]]))
        assert ei.value.code == tb.TB_ERR_CUDA
