"""Parity protocol shared by the -m gpu tests and __graft_entry__.smoke().

Compares the CUDA path (through the C-ABI binding) with the CPU oracle on the same seeded inputs:
  (i)   source indices: bit-exact, except samples whose exact shift lies within 1e-9 of a rounding
        tie (decided by the oracle's extended-precision arbiter) -- those may differ by one; the
        gathered series must be bit-equal;
  (ii)  spectra: |P_gpu - P_orc| <= 1e-4 * max(P_orc, m(k)) (interbinned), and the same with
        max(P^_orc, 1) for the normalised spectrum; the oracle is run on the GPU's indices so that
        an excused tie flip does not masquerade as a spectrum error;
  (iii) harmonic sums (tb_debug_hsums tap, every fold and bin): |S_gpu - S_orc| <= 1e-4 * max(S_orc, 2^L);
  (iv)  candidates: the symmetric set difference holds only entries whose oracle sigma is within
        1e-3 of the threshold; matched entries agree in power (1e-4 * max(S, 2^L)) and sigma (1e-3).

The oracle needs seconds per template at the full sizes, so ``pooled_parity`` runs it in a pool of
worker processes: the main process takes the GPU's outputs through the debug taps, parks them in
/dev/shm, and a worker runs the oracle for that template and does the comparison.
"""
import multiprocessing as mp
import os
import shutil
import tempfile
import threading

import numpy as np

from oracle import tb_oracle as orc

TIE_WINDOW = 1e-9
REL_TOL = 1e-4
SIGMA_BAND = 1e-3
SUMMARY = []                                # one line per full-size comparison, printed by conftest at the end of the run


def compare_indices(idx_gpu, n_samples, tsamp, tmpl, model="bt"):
    idx_orc = orc.resample_indices(n_samples, tsamp, tmpl, model=model)
    mism = np.nonzero(idx_gpu != idx_orc)[0]
    if mism.size:
        assert mism.size <= 8, f"{mism.size} index mismatches (first at j={mism[0]})"
        assert np.all(np.abs(idx_gpu[mism] - idx_orc[mism]) == 1)
        dist = orc.tie_distance(mism, tsamp, tmpl, model)
        assert np.all(dist < TIE_WINDOW), f"index mismatch outside the tie window: j={mism}, dist={dist}"
    return int(mism.size)


def check_indices(plan, wl, tmpl, model="bt"):
    idx_gpu = plan.debug_indices(tmpl)
    return idx_gpu, compare_indices(idx_gpu, wl.n_samples, wl.tsamp, tmpl, model)


WHITE_ATOL = 3e-5                           # |x'_gpu - x'_oracle| of a whitened (unit-variance) series: two fp32 FFTs of length N


def compare_template(series, tsamp, tmpl, tid, W, fill, k_lo, f_min, gpu, sigma_threshold, folds, gpu_cands, kappa=None, model="bt", oversample=False):
    """All comparisons for one template.  gpu: dict with idx, y, P, Ph, med and optionally S
    (float32[5, Nb]).  Returns a small report dict; raises AssertionError on a parity failure.
    kappa: None for the default path (per-template block medians, G15); for a whitened plan (reading
    G25) `series` is the ORACLE's whitened series and kappa the oracle's constant: the gathered
    series may then differ from the GPU's by the rounding of the whitening FFTs (WHITE_ATOL)."""
    n = len(series)
    n_flips = compare_indices(gpu["idx"], n, tsamp, tmpl, model)           # model: "bt" (Kepler solve) or "ell" (plan delay_model=1)
    nb = n if oversample else n // 2                     # spectrum bins (half bins in the oversampled variant G12b)
    if kappa is None:
        spec = orc.spectrum_of_template(series, tsamp, tmpl, W, fill, idx=gpu["idx"], oversample=oversample)
        assert np.array_equal(gpu["y"], spec["resampled"]), "resampled series differs"
        base = orc.median_baseline(spec["medians"], nb, W)
        eM = np.abs(gpu["med"].astype(np.float64) - spec["medians"]) / spec["medians"]
    else:
        spec = orc.spectrum_of_template_whitened(series, kappa, tsamp, tmpl, fill, idx=gpu["idx"])
        dy = np.abs(gpu["y"].astype(np.float64) - spec["resampled"])
        assert dy.max() <= WHITE_ATOL, f"resampled whitened series differs by {dy.max():.3g}"
        base = np.full(nb, orc.LN2 / kappa)
        eM = np.abs(gpu["med"].astype(np.float64) - orc.LN2 / kappa) / (orc.LN2 / kappa)     # the tap reports ln2 / kappa
    eP = np.abs(gpu["P"].astype(np.float64) - spec["power"]) / np.maximum(spec["power"], base)
    eH = np.abs(gpu["Ph"].astype(np.float64) - spec["normalised"]) / np.maximum(spec["normalised"], 1.0)
    assert eP.max() <= REL_TOL, f"interbinned spectrum off by {eP.max():.3g} at bin {eP.argmax()}"
    assert eM.max() <= REL_TOL, f"block median off by {eM.max():.3g} at block {eM.argmax()}"
    assert eH.max() <= REL_TOL, f"normalised spectrum off by {eH.max():.3g} at bin {eH.argmax()}"
    report = {"flips": n_flips, "err_power": float(eP.max()), "err_norm": float(eH.max()), "err_med": float(eM.max())}
    sums = None
    if gpu.get("S") is not None:
        sums = orc.harmonic_sums(spec["normalised"], (0, 1, 2, 3, 4))
        worst = 0.0
        for L in range(5):
            e = np.abs(gpu["S"][L].astype(np.float64) - sums[L]) / np.maximum(sums[L], float(1 << L))
            assert e.max() <= REL_TOL, f"harmonic sum S_{L} off by {e.max():.3g} at bin {e.argmax()}"
            worst = max(worst, float(e.max()))
        report["err_hsum"] = worst
        report["hsum_bins"] = 5 * nb
    if gpu_cands is not None:
        if sums is None or any(L not in sums for L in folds):
            sums = orc.harmonic_sums(spec["normalised"], folds)
        assert k_lo == (orc.lowest_bin_oversampled if oversample else orc.lowest_bin)(n, tsamp, f_min)
        ocand = orc.candidates_from_sums({L: sums[L] for L in folds}, tid, sigma_threshold, k_lo)
        report.update(compare_candidates(gpu_cands, ocand, sums, sigma_threshold))
    return report


def gpu_outputs(plan, tmpl, hsums=False):
    P, Ph, med = plan.debug_spectrum(tmpl)
    out = {"idx": plan.debug_indices(tmpl), "y": plan.debug_resampled(tmpl), "P": P, "Ph": Ph, "med": med}
    if hsums:
        out["S"] = plan.debug_hsums(tmpl)
    return out


def check_template(plan, wl, tid, sigma_threshold=None, folds=None, gpu_cands=None, hsums=False, white=None, model="bt", oversample=False):
    """Full per-template parity in this process; returns a small report dict.
    white: (oracle's whitened series, oracle's kappa) for a plan created with whiten=True."""
    tmpl = wl.templates[tid]
    folds = wl.folds if folds is None else folds
    sigma_threshold = wl.sigma_threshold if sigma_threshold is None else sigma_threshold
    info = plan.info()
    series, kappa = (wl.series, None) if white is None else white
    fill = info["fill_value"] if white is None else orc.fill_value(series)
    return compare_template(series, wl.tsamp, tmpl, tid, plan.median_window, fill, info["k_lo"], wl.f_min,
                            gpu_outputs(plan, tmpl, hsums), sigma_threshold, folds, gpu_cands, kappa, model, oversample)


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
        scale = max(ref[3], float(1 << key[0]))
        worst = max(worst, abs(float(c["power"]) - ref[3]) / scale)
        assert abs(float(c["power"]) - ref[3]) <= REL_TOL * scale
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


# ------------------------------------------------------------------ oracle in a process pool
_CTX = {}                                   # set in the parent before the pool forks: series etc.


def _pool_job(job):
    tid, slot, path, has_s = job
    c = _CTX
    try:
        gpu = {k: np.load(os.path.join(path, f"{k}.npy")) for k in ("idx", "y", "P", "Ph", "med")}
        if has_s:
            gpu["S"] = np.load(os.path.join(path, "S.npy"))
        cands = np.load(os.path.join(path, "cands.npy")) if os.path.exists(os.path.join(path, "cands.npy")) else None
        rep = compare_template(c["series"], c["tsamp"], c["templates"][tid], slot, c["W"], c["fill"], c["k_lo"], c["f_min"],
                               gpu, c["sigma"], c["folds"], cands, c["kappa"], c["model"])
        return tid, rep, None
    except AssertionError as e:
        return tid, None, f"template {tid}: {e}"
    finally:
        shutil.rmtree(path, ignore_errors=True)


def default_workers(n_samples):
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        cores = os.cpu_count() or 1
    per_worker_gb = 200.0 * n_samples / 2**30          # ~25 fp64 arrays of N live at the oracle's peak
    try:
        avail_gb = os.sysconf("SC_AVPHYS_PAGES") * os.sysconf("SC_PAGE_SIZE") / 2**30
    except (ValueError, OSError):
        avail_gb = 32.0
    return int(max(1, min(cores, 32, 0.6 * avail_gb / max(per_worker_gb, 1e-3))))


def pooled_parity(plan, wl, ids, sigma_threshold, folds, per_cands, hsums_ids=(), slots=None, workers=None, white=None, model="bt"):
    """check_template for many templates with the oracle in a pool of forked workers.
    ids: template indices into wl.templates; per_cands: {slot id -> candidate rows} of the GPU (a
    template without an entry is compared against an empty list); slots: the template_id each of
    `ids` carries in the candidate list (default: the index itself).  Returns {id: report}."""
    ids = list(ids)
    slots = dict(zip(ids, ids if slots is None else slots))
    info = plan.info()
    _CTX.clear()
    series, kappa = (wl.series, None) if white is None else white
    _CTX.update(series=series, tsamp=wl.tsamp, templates=wl.templates, W=plan.median_window,
                fill=info["fill_value"] if white is None else orc.fill_value(series), kappa=kappa, model=model,
                k_lo=info["k_lo"], f_min=wl.f_min, sigma=sigma_threshold, folds=tuple(folds))
    workers = workers or default_workers(wl.n_samples)
    shm = "/dev/shm" if os.path.isdir("/dev/shm") else None
    root = tempfile.mkdtemp(prefix="tb_parity_", dir=shm)
    gate = threading.Semaphore(2 * workers)             # GPU outputs parked at once
    reports, errors = {}, []

    def done(res):
        tid, rep, err = res
        if err:
            errors.append(err)
        else:
            reports[tid] = rep
        gate.release()

    def failed(exc):
        errors.append(repr(exc))
        gate.release()

    empty = np.zeros(0, dtype=[("template_id", "<u4"), ("fold", "<u4"), ("bin", "<u4"), ("power", "<f4"), ("sigma", "<f4"), ("pad", "<u4")])
    try:
        with mp.get_context("fork").Pool(workers) as pool:
            for tid in ids:
                gate.acquire()
                if errors:
                    gate.release()
                    break
                has_s = tid in hsums_ids
                out = gpu_outputs(plan, wl.templates[tid], has_s)
                path = os.path.join(root, str(tid))
                os.makedirs(path)
                for k, v in out.items():
                    np.save(os.path.join(path, f"{k}.npy"), v)
                if per_cands is not None:
                    np.save(os.path.join(path, "cands.npy"), per_cands.get(slots[tid], empty))
                pool.apply_async(_pool_job, ((tid, slots[tid], path, has_s),), callback=done, error_callback=failed)
            pool.close()
            pool.join()
    finally:
        shutil.rmtree(root, ignore_errors=True)
    assert not errors, "; ".join(errors[:5])
    assert len(reports) == len(ids)
    return reports
