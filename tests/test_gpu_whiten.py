"""-m gpu: the whitened mode (opts.whiten, reading G25) against the oracle's
whiten_series / whitened_level / search_template_whitened.  The oracle whitens the series itself
(no oracle input comes from the CUDA path): the two whitened series differ by the rounding of two
fp32 FFTs (3e-5 of a unit-variance series), everything after that by the usual 1e-4."""
import numpy as np
import pytest

from oracle import tb_oracle as orc
from paper_2112_11991_b200 import workloads as wl_mod

from parity import SUMMARY, WHITE_ATOL, by_template, check_template, pooled_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tb():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2112_11991_b200 import build
    build.build()
    from paper_2112_11991_b200 import tb
    return tb


def _whitened_oracle(series, window=1024, zap=()):
    xw = orc.whiten_series(series, window, zap)
    return xw, orc.whitened_level(xw, window, zap)


def _check_series(plan, xw, kappa):
    xg, kg = plan.debug_series()
    d = np.abs(xg.astype(np.float64) - xw)
    assert d.max() <= WHITE_ATOL, f"whitened series differs by {d.max():.3g} at {d.argmax()}"
    assert abs(kg / kappa - 1.0) < 1e-5
    assert plan.info()["fill_value"] == pytest.approx(float(orc.fill_value(xw)), abs=1e-6)
    return float(d.max())


def test_c1_whitened_full_parity(tb, c1):
    xw, kappa = _whitened_oracle(c1.series)
    with tb.Plan(c1.series, c1.tsamp, whiten=True) as plan:
        err_x = _check_series(plan, xw, kappa)
        plan.search(c1.templates, 0, c1.folds, 6.0)
        cands, n = plan.candidates()
        per = by_template(cands)
        rep = pooled_parity(plan, c1, range(len(c1.templates)), 6.0, c1.folds, per, hsums_ids=range(0, 64, 8), white=(xw, kappa))
    assert set(per) == {0}
    best = cands[np.argmax(cands["sigma"])]
    assert (int(best["fold"]), int(best["bin"])) == (3, 52429)
    o = orc.search_template_whitened(xw, kappa, c1.tsamp, c1.templates[0])
    assert sum(r["n_oracle"] for r in rep.values()) == len(o)
    SUMMARY.append(f"C1 whitened sigma 6: {n} candidates, 64 templates compared; whitened series off by {err_x:.2g}, "
                   f"worst spectrum error {max(r['err_norm'] for r in rep.values()):.2g}")


def test_whitening_of_red_noise_and_zapping(tb):
    """A red series with a strong interference tone: whitened + zapped on the device as in the oracle;
    without the zap the tone is found by every template, with it by none."""
    rng = np.random.default_rng(77)
    n, tsamp, k0 = 1 << 18, 1e-3, 20000
    w = rng.standard_normal(n)
    x = (np.cumsum(w) * 0.02 + w + 0.1 * np.cos(2 * np.pi * k0 * np.arange(n) / n)).astype(np.float32)
    wl = wl_mod.Workload("red", n, tsamp, x, np.array([[150.0, 0.0, 0.0, 0.0, 0.0], [90.0, 0.02, 1.0, 0.0, 0.0]]), (), ())
    zap = [(k0 - 2, k0 + 3)]
    xw, kappa = _whitened_oracle(x, zap=zap)
    with tb.Plan(x, tsamp, whiten=True, zap_ranges=zap) as plan:
        _check_series(plan, xw, kappa)
        plan.search(wl.templates, 0, wl.folds, 7.0)
        cands, _ = plan.candidates()
        for tid in (0, 1):
            check_template(plan, wl, tid, 7.0, wl.folds, by_template(cands).get(tid, cands[:0]), hsums=True, white=(xw, kappa))
        zapped = cands
    with tb.Plan(x, tsamp, whiten=True) as plan:
        plan.search(wl.templates[:1], 0, wl.folds, 7.0)
        kept, _ = plan.candidates()

    def at_tone(c):                                              # fold-0 detections within 3 bins of the tone
        return int(np.count_nonzero((c["fold"] == 0) & (np.abs(c["bin"].astype(np.int64) - k0) <= 3)))
    # (the steep bottom of the random-walk spectrum, below the first block centre where the baseline
    # is flat, leaves low-frequency detections in both runs: they are compared with the oracle above)
    assert at_tone(kept) >= 1 and at_tone(zapped) == 0


@pytest.mark.parametrize("log2n,window,fft_path", [(12, 256, 0), (17, 256, 2), (17, 1024, 1), (20, 512, 2), (23, 1024, 2), (24, 2048, 2)])
def test_whitened_both_paths_and_windows(tb, log2n, window, fft_path):
    w = wl_mod.config1() if log2n <= 17 else wl_mod.config5(log2n=log2n)
    if log2n == 12:
        w = wl_mod.Workload("tiny", 4096, 1e-3, w.series[:4096].copy(), np.array([[3.0, 0.05, 0.5, 0.0, 0.0], [2.5, 0.04, 2.0, 0.3, 1.0]]), (), ())
    xw, kappa = _whitened_oracle(w.series, window)
    ids = [0, 1] if log2n <= 17 else [3, 256 + 5]
    with tb.Plan(w.series, w.tsamp, median_window=window, fft_path=fft_path, whiten=True) as plan:
        _check_series(plan, xw, kappa)
        plan.search(w.templates[ids], 0, w.folds, 5.0)
        cands, n = plan.candidates()
        rep = pooled_parity(plan, w, ids, 5.0, w.folds, by_template(cands), hsums_ids=ids, slots=[0, 1], white=(xw, kappa))
    assert all("err_hsum" in r for r in rep.values())


def test_wide_birdie_list_does_not_inflate_kappa(tb, c1):
    """6 % of the band zapped (whole blocks, a straddle, a part of a block; reading G25): the device's kappa is the
    oracle's -- both leave the touched blocks out of the mean -- and stays within 1.5 % of the unzapped series'
    kappa instead of growing by 1 / (1 - 0.06); candidates equal the oracle's on the true template."""
    W = 1024
    zap = [(8 * W, 10 * W), (30 * W + 100, 31 * W + 900), (50 * W, 50 * W + 300)]
    xw, kappa = _whitened_oracle(c1.series, W, zap)
    with tb.Plan(c1.series, c1.tsamp, whiten=True, zap_ranges=zap) as plan:
        _check_series(plan, xw, kappa)
        kg = plan.debug_series()[1]
        plan.search(c1.templates[:2], 0, c1.folds, 6.0)
        cands, _ = plan.candidates()
        for tid in (0, 1):
            check_template(plan, c1, tid, 6.0, c1.folds, by_template(cands).get(tid, cands[:0]), hsums=True, white=(xw, kappa))
    with tb.Plan(c1.series, c1.tsamp, whiten=True) as plan:
        k0 = plan.debug_series()[1]
    assert abs(kg / k0 - 1.0) < 0.015
    assert orc.whitened_level(xw, W) / kappa > 1.04              # what the round-2 rule (every block) would give


def test_set_series_rewhitens(tb, c1):
    other = np.random.default_rng(5).standard_normal(c1.n_samples).astype(np.float32) * 2.0 + 1.0
    with tb.Plan(other, c1.tsamp, whiten=True) as plan:
        plan.set_series(c1.series)
        _check_series(plan, *_whitened_oracle(c1.series))


def test_bench_config_whitened(tb):
    """bench.py's workload (C5 at 2^23) in the whitened mode: 16 templates compared in full."""
    w = wl_mod.config5(log2n=23)
    xw, kappa = _whitened_oracle(w.series)
    ids = list(range(0, 256, 32)) + list(range(256, 512, 32))
    with tb.Plan(w.series, w.tsamp, whiten=True) as plan:
        err_x = _check_series(plan, xw, kappa)
        plan.search(w.templates, 0, w.folds, 4.5)
        cands, n = plan.candidates()
        rep = pooled_parity(plan, w, ids, 4.5, w.folds, by_template(cands), hsums_ids=ids[::4], white=(xw, kappa))
    SUMMARY.append(f"C5/2^23 whitened sigma 4.5: {n} candidates in 512 templates, {len(ids)} compared; whitened series off by "
                   f"{err_x:.2g}, worst spectrum error {max(r['err_norm'] for r in rep.values()):.2g}, "
                   f"in the threshold band {sum(r['n_band'] for r in rep.values())}")
