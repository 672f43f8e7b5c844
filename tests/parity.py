"""Parity protocol shared by the -m gpu tests and __graft_entry__.smoke().

Compares the CUDA path (through the C-ABI binding) with the CPU oracle on the same seeded inputs:
  (i)   source indices: bit-exact, except samples whose exact shift lies within 1e-9 of a rounding
        tie (decided by the oracle's extended-precision arbiter) -- those may differ by one;
  (ii)  spectra: |P_gpu - P_orc| <= 1e-4 * max(P_orc, m(k)) (interbinned), and the same with
        max(P^_orc, 1) for the normalised spectrum; the oracle is run on the GPU's indices so that
        an excused tie flip does not masquerade as a spectrum error;
  (iii) candidates: the symmetric set difference holds only entries whose oracle sigma is within
        1e-3 of the threshold.
"""
import numpy as np

from oracle import tb_oracle as orc

TIE_WINDOW = 1e-9
REL_TOL = 1e-4
SIGMA_BAND = 1e-3


def check_indices(plan, wl, tmpl):
    idx_gpu = plan.debug_indices(tmpl)
    idx_orc = orc.resample_indices(wl.n_samples, wl.tsamp, tmpl)
    mism = np.nonzero(idx_gpu != idx_orc)[0]
    if mism.size:
        assert mism.size <= 8, f"{mism.size} index mismatches (first at j={mism[0]})"
        assert np.all(np.abs(idx_gpu[mism] - idx_orc[mism]) == 1)
        dist = orc.tie_distance(mism, wl.tsamp, tmpl)
        assert np.all(dist < TIE_WINDOW), f"index mismatch outside the tie window: j={mism}, dist={dist}"
    return idx_gpu, int(mism.size)


def check_template(plan, wl, tid, sigma_threshold=None, folds=None, gpu_cands=None):
    """Full per-template parity; returns a small report dict."""
    tmpl = wl.templates[tid]
    folds = wl.folds if folds is None else folds
    sigma_threshold = wl.sigma_threshold if sigma_threshold is None else sigma_threshold
    W = plan.median_window
    info = plan.info()
    idx_gpu, n_flips = check_indices(plan, wl, tmpl)
    spec = orc.spectrum_of_template(wl.series, wl.tsamp, tmpl, W, info["fill_value"], idx=idx_gpu)
    y = plan.debug_resampled(tmpl)
    assert np.array_equal(y, spec["resampled"]), "resampled series differs"
    P, Ph, med = plan.debug_spectrum(tmpl)
    nb = wl.n_samples // 2
    base = orc.median_baseline(spec["medians"], nb, W)
    eP = np.abs(P.astype(np.float64) - spec["power"]) / np.maximum(spec["power"], base)
    eH = np.abs(Ph.astype(np.float64) - spec["normalised"]) / np.maximum(spec["normalised"], 1.0)
    eM = np.abs(med.astype(np.float64) - spec["medians"]) / spec["medians"]
    assert eP.max() <= REL_TOL, f"interbinned spectrum off by {eP.max():.3g} at bin {eP.argmax()}"
    assert eM.max() <= REL_TOL, f"block median off by {eM.max():.3g} at block {eM.argmax()}"
    assert eH.max() <= REL_TOL, f"normalised spectrum off by {eH.max():.3g} at bin {eH.argmax()}"
    report = {"flips": n_flips, "err_power": float(eP.max()), "err_norm": float(eH.max()), "err_med": float(eM.max())}
    if gpu_cands is not None:
        sums = orc.harmonic_sums(spec["normalised"], folds)
        k_lo = orc.lowest_bin(wl.n_samples, wl.tsamp, wl.f_min)
        assert k_lo == info["k_lo"]
        ocand = orc.candidates_from_sums(sums, tid, sigma_threshold, k_lo)
        report.update(compare_candidates(gpu_cands, ocand, sums, sigma_threshold))
    return report


def compare_candidates(gpu_cands, ocand, sums, sigma_threshold):
    """gpu_cands: structured array rows of ONE template; ocand: oracle list for the same template."""
    g = {(int(c["fold"]), int(c["bin"])): c for c in gpu_cands}
    o = {(c[1], c[2]): c for c in ocand}
    for key in set(g) ^ set(o):
        L, k = key
        sig = float(orc.sigma_of_power(sums[L][k], L))
        assert abs(sig - sigma_threshold) <= SIGMA_BAND, \
            f"candidate (fold {L}, bin {k}) in {'gpu' if key in g else 'oracle'} only; oracle sigma {sig}"
    worst = 0.0
    for key in set(g) & set(o):
        c, ref = g[key], o[key]
        worst = max(worst, abs(float(c["power"]) - ref[3]) / max(ref[3], 1.0))
        assert abs(float(c["power"]) - ref[3]) <= 2 * REL_TOL * max(ref[3], 1.0) * (1 << key[0]) ** 0.5
        assert abs(float(c["sigma"]) - ref[4]) <= 1e-3
    return {"n_gpu": len(g), "n_oracle": len(o), "n_band": len(set(g) ^ set(o)), "err_cand_power": worst}


def by_template(cands):
    """Split a sorted candidate array into {template_id: rows}."""
    out = {}
    if len(cands):
        ids = cands["template_id"]
        cuts = np.nonzero(np.diff(ids))[0] + 1
        for part in np.split(cands, cuts):
            out[int(part["template_id"][0])] = part
    return out
