"""-m gpu: the 2x-oversampled interbinning variant (reading G12b; plan option
interbin_oversample) against the oracle's interbin_power_oversampled, element by element: spectra of
N half bins, block medians, every harmonic sum and the candidate list, through the same protocol and
tolerances as the default spectrum (tests/parity.py)."""
import numpy as np
import pytest

from oracle import tb_oracle as orc
from paper_2112_11991_b200 import workloads as wl_mod

from parity import by_template, check_template

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tb():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2112_11991_b200 import build
    build.build()
    from paper_2112_11991_b200 import tb
    return tb


def test_c1_oversampled_full_parity(tb, c1):
    with tb.Plan(c1.series, c1.tsamp, interbin_oversample=True, enable_timings=True) as plan:
        assert plan.info()["k_lo"] == orc.lowest_bin_oversampled(c1.n_samples, c1.tsamp, c1.f_min)
        plan.search(c1.templates[:16], 0, c1.folds, 5.0)
        assert plan.timings()["fft_path_used"] == 1                  # library-FFT path
        cands, n = plan.candidates()
        per = by_template(cands)
        assert 0 in per and cands["bin"].max() < c1.n_samples
        best = cands[np.argmax(cands["sigma"])]
        f = best["bin"] / (2.0 * (1 << int(best["fold"])) * c1.t_obs)                 # half bins
        assert int(best["template_id"]) == 0 and abs(f - 50.0) < 1.0 / c1.t_obs
        worst = 0.0
        for tid in range(16):
            rep = check_template(plan, c1, tid, 5.0, c1.folds, per.get(tid, cands[:0]), hsums=tid in (0, 5), oversample=True)
            worst = max(worst, rep["err_norm"], rep["err_power"], rep.get("err_hsum", 0.0))
            assert rep["n_gpu"] == rep["n_oracle"] or rep["n_band"] > 0
        assert worst <= 1e-4
        print(f"oversampled C1: {n} candidates, worst relative error {worst:.2g}")


@pytest.mark.parametrize("log2n,window", [(13, 256), (20, 2048)])
def test_oversampled_windows_and_elliptical(tb, log2n, window):
    w = wl_mod.config5(log2n=log2n) if log2n >= 20 else None
    if w is None:
        x = np.random.default_rng(3).standard_normal(1 << log2n).astype(np.float32)
        w = wl_mod.Workload("tiny", 1 << log2n, 1e-3, x, np.array([[3.0, 0.05, 0.5, 0.0, 0.0], [2.5, 0.04, 2.0, 0.3, 1.0]]), (), ())
        ids = [0, 1]
    else:
        ids = [7, 256 + 9]
    with tb.Plan(w.series, w.tsamp, interbin_oversample=True, median_window=window) as plan:
        plan.search(w.templates[ids], 0, w.folds, 4.5)
        cands, _ = plan.candidates()
        per = by_template(cands)
        ww = type(w)(w.name, w.n_samples, w.tsamp, w.series, w.templates[ids], (), ())
        for slot in range(2):
            rep = check_template(plan, ww, slot, 4.5, w.folds, per.get(slot, cands[:0]), hsums=True, oversample=True)
            assert rep["err_hsum"] <= 1e-4


def test_scalloped_tone_is_recovered(tb):
    """A sinusoid midway between two bins: the odd half bin carries (pi/2)^2 of the raw bins' power."""
    n, tsamp = 1 << 14, 1e-3
    j = np.arange(n)
    x = (np.random.default_rng(8).standard_normal(n) + 0.12 * np.cos(2 * np.pi * 1000.5 * j / n)).astype(np.float32)
    tmpl = np.array([[50.0, 0.0, 0.0, 0.0, 0.0]])
    with tb.Plan(x, tsamp, interbin_oversample=True) as plan:
        plan.search(tmpl, 0, (0,), 5.0)
        cands, _ = plan.candidates()
        P, Ph, med = plan.debug_spectrum(tmpl[0])
    assert P.size == n and med.size == n // 1024
    assert int(cands[np.argmax(cands["sigma"])]["bin"]) == 2001
    assert P[2001] > 1.8 * max(P[2000], P[2002])
    ref = orc.search_template(x, tsamp, tmpl[0], 0, (0,), 5.0, oversample=True)
    assert [(c[1], c[2]) for c in ref] == [(int(c["fold"]), int(c["bin"])) for c in cands]


def test_oversample_option_combinations(tb, c1):
    for kw in [dict(fft_path=2), dict(whiten=True)]:
        with pytest.raises(tb.TbError) as ei:
            tb.Plan(c1.series, c1.tsamp, interbin_oversample=True, **kw)
        assert ei.value.code == tb.TB_ERR_INVALID_ARG
