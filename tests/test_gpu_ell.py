"""-m gpu: the ELL7 approximate-orbit resampler (opts.delay_model = 1, reading G26)
against the oracle's roemer_delay_ell: indices bit-exact outside the 1e-9 tie window (arbiter: the
same series in extended precision), spectra / harmonic sums / candidates as for the default mode."""
import numpy as np
import pytest

from oracle import tb_oracle as orc
from paper_2112_11991_b200 import workloads as wl_mod

from parity import SUMMARY, by_template, check_indices, pooled_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tb():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2112_11991_b200 import build
    build.build()
    from paper_2112_11991_b200 import tb
    return tb


def test_ell_small_full_parity(tb):
    w = wl_mod.config4(n_templates=24, log2n=18, tau_scale=1.0 / 128)
    with tb.Plan(w.series, w.tsamp, delay_model=1) as plan:
        plan.search(w.templates, 0, w.folds, 5.0)
        cands, n = plan.candidates()
        per = by_template(cands)
        rep = pooled_parity(plan, w, range(24), 5.0, w.folds, per, hsums_ids=range(0, 24, 6), model="ell")
    assert 0 in per                                               # e = 0.08: the ELL7 orbit still finds the injected pulsar
    assert max(r["flips"] for r in rep.values()) <= 2


def test_ell_indices_high_eccentricity_and_exact_fallback(tb, c1):
    """Index parity where the series visibly departs from the Kepler solve (e = 0.3: whole samples) and
    for orbits too fast to interpolate (knot spacing < 8: every sample from the series itself)."""
    with tb.Plan(c1.series, c1.tsamp, delay_model=1) as plan, tb.Plan(c1.series, c1.tsamp) as bt:
        for tmpl in [(60.0, 0.5, 1.0, 0.05, 0.7), (45.0, 0.8, 2.0, 0.3, 4.0), (0.5, 0.02, 1.0, 0.1, 2.0), (3.0, 0.2, 0.1, 0.1, 0.3),
                     (400.0, 20.0, 0.9, 0.3, 0.7)]:
            idx, flips = check_indices(plan, c1, np.array(tmpl), model="ell")
            assert flips <= 2
        d = np.abs(idx - bt.debug_indices(np.array(tmpl)))         # e = 0.3, tau/tsamp = 2e4: 1.2 e^7 tau/tsamp = 5 samples
        assert 2 <= d.max() <= 8
        assert plan.knot_log2((0.5, 0.02, 1.0, 0.1, 2.0)) <= 2


def test_ell_c4_full_size(tb):
    """C4 (2^23, e <= 0.1, tau up to 8 lt-s) in the ELL7 mode: the true template and 15 sampled ones."""
    w = wl_mod.config4()
    ids = [0] + [int(i) for i in np.random.default_rng(4).choice(np.arange(1, 8192), 15, replace=False)]
    with tb.Plan(w.series, w.tsamp, delay_model=1, enable_timings=True) as plan:
        plan.search(w.templates[:512], 0, w.folds, 6.0)
        t = plan.timings()
        cands, n = plan.candidates()
        per = by_template(cands)
        plan.search(w.templates[ids], 0, w.folds, 6.0)
        sub, _ = plan.candidates()
        rep = pooled_parity(plan, w, ids, 6.0, w.folds, by_template(sub), hsums_ids=ids[:2], slots=list(range(len(ids))), model="ell")
    assert 0 in per and t["fft_path_used"] == 2
    SUMMARY.append(f"C4 ELL7 mode sigma 6: 512 templates searched ({t['ms_delay'] / 512 * 1e3:.2f} us per template in the knot kernel), "
                   f"{len(ids)} compared; index flips {sum(r['flips'] for r in rep.values())}, worst spectrum error "
                   f"{max(r['err_norm'] for r in rep.values()):.2g}")


def test_invalid_delay_model(tb, c1):
    with pytest.raises(tb.TbError) as ei:
        tb.Plan(c1.series, c1.tsamp, delay_model=2)
    assert ei.value.code == tb.TB_ERR_INVALID_ARG
