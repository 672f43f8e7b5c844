"""CPU oracle for the template-bank binary-pulsar search hot path (arXiv:2112.11991).

TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, obviously-correct statement of what
the hot path computes.  Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may import it.  It shares no code with
``paper_2112_11991_b200/`` (the CUDA path) and imports nothing from it; the CUDA path never
imports this file.  Inputs come from the caller (the seeded generators live in
``paper_2112_11991_b200/workloads.py`` and contain none of this arithmetic).

Every function cites the passage of ``/root/reference/PAPER.md`` it follows (``PAPER.md:L<n>``)
and, where the paper is silent, the reading of SURVEY.md §8(c) / DESIGN.md §3 (``G<n>``).

Arithmetic: fp64 (numpy) after loading the float32 series.  One deliberate exception
(reading G10): where the fp64 shift lies within ``TIE_GUARD`` of a rounding tie the
shift is re-evaluated with the *same formulas* in x87 extended precision (``numpy.longdouble``,
64-bit mantissa) so that the integer decision is that of the exact real-number formula to far
better than the 1e-9-sample tie window the north_star allows.

Parity pins (tests/test_oracle_pins.py, ``-m "not gpu"``):
  kepler_solve ............ T4  residual <= 1e-12 and the printed App. B series
  roemer_delay ............ T2  e=0 Kepler path == circular closed form; T1 tau=0 -> identity;
                            e>0: eq A1 assembled from the PRINTED e-series (eqs 15-16, App. B) to
                            2 e^7 tau, and the hand-solvable points M = 0, pi, pi/2 - e
  resample_indices ........ T1, T3 (idx_0 = 0), T11 (monotone map, out-of-range bound); the
                            extended-precision re-decision: samples built 2e-11..3e-8 from a
                            rounding tie against a 50-digit mpmath evaluation (both sides)
  sign convention (G2-G4) . a series synthesised from eq A2 read literally (t' = t - Delta_R(t),
                            no inverse map) is found at phi0 + pi and not at phi0: the paper is
                            at odds with itself about this sign (eq 2/4 vs A2 vs Alg. 1), so
                            the reading is pinned only up to that phase flip (both are searched)
  rfft_forward ............ T5 Parseval, T6 brute-force O(N^2) DFT at N=1024
  interbin_power .......... T7 closed forms for an integer-bin and a half-bin tone
  block_medians / baseline  hand-sorted toy input; T8 median = ln2 * mean for exponential noise
  harmonic_sums ........... T6 direct double loop from eq 9; comb of tones -> S_4[16 k0] = 16 P
  sigma constants ......... T9 equals eq 11 at n=1 (printed constants sqrt(pi/4), sqrt(1-pi/4))
  search (end to end) ..... T10 injected pulsar found with its true template at its spin
                            frequency, not found without resampling
  Parity UNPINNED by the paper (north_star / SURVEY proposal only; pinned solely by closed
  forms T7/T8): the choice of interbinning formula (G12), the block-median estimator (G15),
  f_min (G20) and the out-of-range fill value (G8).
"""
from __future__ import annotations

import math
from typing import Iterable, Sequence

import numpy as np

LN2 = math.log(2.0)
TIE_GUARD = 1e-6          # |frac(delta) - 1/2| below this -> decide in extended precision (G10)
KEPLER_TOL = 1e-12        # rad, BASELINE.json C4 "Newton Kepler solve to 1e-12 rad" (G9)
KEPLER_MAX_ITER = 50


# ----------------------------------------------------------------------------------------------
# O1/O2  orbit model
# ----------------------------------------------------------------------------------------------
def _two_pi(dtype):
    """2*pi in the working precision (numpy.pi is only a double)."""
    return dtype(8) * np.arctan(dtype(1))


def kepler_solve(M, e, tol=KEPLER_TOL, max_iter=KEPLER_MAX_ITER):
    """Eccentric anomaly E with E - e sin E = M (eq 3; Alg. 1).

    The paper says only "solve for E iteratively"; reading G9: Newton's method started at
    E0 = M + e sin M, iterated until every |dE| <= tol (1e-12 rad) or ``max_iter`` steps.
    Works elementwise on arrays, in the dtype of ``M`` (float64 or longdouble).
    """
    M = np.asarray(M)
    e = M.dtype.type(e)
    E = M + e * np.sin(M)
    for _ in range(max_iter):
        dE = (E - e * np.sin(E) - M) / (1 - e * np.cos(E))
        E = E - dE
        if dE.size == 0 or np.max(np.abs(dE)) <= tol:
            break
    return E


def is_circular(tmpl) -> bool:
    """A template with e == 0 and omega == 0 uses the circular closed form (eq 4 = eq A1
    L666 at e = 0, omega = 0).  The library's own selector is e == 0 alone (include/tb.h: E = M, Delta =
    tau sin(Omega t + phi0 + omega)); at e = 0 and omega != 0 this oracle goes through eq A1 with the Newton
    solve, which returns E = M exactly there, so the two agree (reading G6)."""
    return float(tmpl[3]) == 0.0 and float(tmpl[4]) == 0.0


# Appendix B of the paper: coefficients of the e-series of eqs 15-16 (L106-111),
#   cos E = sum_k C_k(e) cos kM,   sqrt(1 - e^2) sin E = sum_k S_k(e) sin kM,
# as {k: ((power of e, numerator, denominator), ...)}, "up-to the 7th power in e" = terms through e^6
# of the ELL7 model (L668).  tests/test_oracle_pins.py checks this table against the same numbers
# typed independently into tests/golden/appendix_b_series.txt.
ELL_C = {0: ((1, -1, 2),),
         1: ((0, 1, 1), (2, -3, 8), (4, 5, 192), (6, -7, 9216)),
         2: ((1, 1, 2), (3, -1, 3), (5, 1, 16)),
         3: ((2, 3, 8), (4, -45, 128), (6, 567, 5120)),
         4: ((3, 1, 3), (5, -2, 5)),
         5: ((4, 125, 384), (6, -4375, 9216)),
         6: ((5, 27, 80),),
         7: ((6, 16807, 46080),)}
ELL_S = {1: ((0, 1, 1), (2, -5, 8), (4, -11, 192), (6, -457, 9216)),
         2: ((1, 1, 2), (3, -5, 12), (5, 1, 24)),
         3: ((2, 3, 8), (4, -51, 128), (6, 543, 5120)),
         4: ((3, 1, 3), (5, -13, 30)),
         5: ((4, 125, 384), (6, -4625, 9216)),
         6: ((5, 27, 80),),
         7: ((6, 16807, 46080),)}


def ell_coefficients(ecc, dtype=np.float64):
    """(C_k(e), k = 0..7), (S_k(e), k = 1..7) of Appendix B as arrays of `dtype`."""
    e = dtype(float(ecc))
    C = [sum(dtype(num) / dtype(den) * e ** pw for pw, num, den in ELL_C[k]) for k in range(8)]
    S = [sum(dtype(num) / dtype(den) * e ** pw for pw, num, den in ELL_S[k]) for k in range(1, 8)]
    return C, S


def roemer_delay_ell(j, tsamp, tmpl, dtype=np.float64):
    """SURVEY 8(f) row f4, reading G26: the ELL7 approximate-orbit delay.  Eq A1 with
    cos E and sqrt(1-e^2) sin E replaced by the printed series of eqs 15-16 (L106-111, L668: "The
    alternative is to expand cos E and sin E as a power series ... ELL1 ... ELL2 and so on"):
        Delta = tau[(sum_{k=0}^{7} C_k cos kM - e) sin(omega) + (sum_{k=1}^{7} S_k sin kM) cos(omega)],
    M = Omega t + phi0.  No Kepler solve.  Differs from the BT delay by about 1.2 e^7 tau."""
    p_orb, tau, phi0, ecc, omega = (dtype(float(v)) for v in tmpl)
    t = np.asarray(j).astype(dtype) * dtype(float(tsamp))
    M = (_two_pi(dtype) / p_orb) * t + phi0
    C, S = ell_coefficients(float(tmpl[3]), dtype)
    cosE = sum(C[k] * np.cos(dtype(k) * M) for k in range(8))
    qsinE = sum(S[k - 1] * np.sin(dtype(k) * M) for k in range(1, 8))
    return tau * ((cosE - ecc) * np.sin(omega) + qsinE * np.cos(omega))


def roemer_delay(j, tsamp, tmpl, dtype=np.float64, force_kepler=False, model="bt"):
    """Roemer delay Delta_R(t = j*tsamp) in seconds.

    tmpl = (P_orb [s], tau = a sin(i)/c [lt-s], phi0 [rad], e, omega [rad]); the paper's
    (alpha, psi) are BASELINE's (phi0, omega).
      M   = Omega t + phi0,  Omega = 2 pi / P_orb            (eq 3; Alg. 1, reading G1)
      circular:   Delta = tau sin(M)                         (eq A1 L666 at e = 0, psi = 0; G6)
      elliptical: Delta = tau[(cos E - e) sin(omega) + sqrt(1-e^2) sin E cos(omega)]   (eq A1)
    model = "bt" (the paper's resampler, L668: "we implemented the BT model") or "ell" (roemer_delay_ell).
    """
    if model == "ell":
        return roemer_delay_ell(j, tsamp, tmpl, dtype)
    p_orb, tau, phi0, ecc, omega = (dtype(float(v)) for v in tmpl)
    t = np.asarray(j).astype(dtype) * dtype(float(tsamp))
    M = (_two_pi(dtype) / p_orb) * t + phi0
    if is_circular(tmpl) and not force_kepler:
        return tau * np.sin(M)
    E = kepler_solve(M, ecc)
    return tau * ((np.cos(E) - ecc) * np.sin(omega) + np.sqrt(1 - ecc * ecc) * np.sin(E) * np.cos(omega))


def shift_in_samples(j, tsamp, tmpl, dtype=np.float64, force_kepler=False, model="bt"):
    """delta_j = (Delta_R(j tsamp) - Delta_R(0)) / tsamp  (zero offset t0: PAPER.md:L675,
    Alg. 1; sign reading G2: the offset is subtracted from the delay so delta_0 = 0)."""
    d = roemer_delay(j, tsamp, tmpl, dtype, force_kepler, model)
    d0 = roemer_delay(np.zeros(1, dtype=np.int64), tsamp, tmpl, dtype, force_kepler, model)[0]
    return (d - d0) / dtype(float(tsamp))


def tie_distance(j, tsamp, tmpl, model="bt"):
    """Arbiter: |frac(delta_j) - 1/2| evaluated in extended precision for the sample numbers j."""
    d = shift_in_samples(np.asarray(j, dtype=np.int64), tsamp, tmpl, np.longdouble, model=model)
    return np.abs((d - np.floor(d)) - np.longdouble(0.5)).astype(np.float64)


def resample_indices(n_samples, tsamp, tmpl, force_kepler=False, model="bt"):
    """idx_j = j - floor(delta_j + 1/2), j = 0..N-1  (Alg. 1 "[.]_int", prose L675
    "nearest integer"; readings G3 = gather evaluated at the output index, G7 = round delta,
    never j - delta).  Returns int64[N]; entries may lie outside [0, N)."""
    j = np.arange(int(n_samples), dtype=np.int64)
    d = shift_in_samples(j, tsamp, tmpl, np.float64, force_kepler, model)
    s = np.floor(d + 0.5).astype(np.int64)
    near = np.abs((d - np.floor(d)) - 0.5) < TIE_GUARD
    if near.any():
        dl = shift_in_samples(j[near], tsamp, tmpl, np.longdouble, force_kepler, model)
        s[near] = np.floor(dl + np.longdouble(0.5)).astype(np.int64)
    return j - s


# ----------------------------------------------------------------------------------------------
# O4  gather
# ----------------------------------------------------------------------------------------------
def fill_value(series) -> np.float32:
    """Value for output samples whose source index is out of range: the series mean, summed in
    fp64, rounded to float32 (paper silent; reading G8)."""
    return np.float32(np.mean(np.asarray(series, dtype=np.float64)))


def gather(series, idx, fill):
    """y_j = x[idx_j] if 0 <= idx_j < N else fill  (Alg. 1; G8).  float32 out."""
    x = np.asarray(series, dtype=np.float32)
    ok = (idx >= 0) & (idx < x.size)
    y = np.full(idx.size, np.float32(fill), dtype=np.float32)
    y[ok] = x[idx[ok]]
    return y


# ----------------------------------------------------------------------------------------------
# O5/O6  spectrum
# ----------------------------------------------------------------------------------------------
def rfft_forward(y):
    """X_k = sum_j y_j exp(-2 pi i j k / N), k = 0..N/2, unnormalised forward transform in fp64
    ("calculate an FFT", L706; G11).  Library FFT is the step itself."""
    return np.fft.rfft(np.asarray(y, dtype=np.float64))


def interbin_power(X):
    """P_k = max(|X_k|^2, 1/2 |X_k - X_{k-1}|^2), k = 0..Nb-1, Nb = N/2, with X_0 <- 0 first and
    X_{-1} = 0; the Nyquist bin is dropped (paper silent: readings G12, G13, G14)."""
    X = np.array(X, dtype=np.complex128)
    nb = X.size - 1
    X[0] = 0.0
    Xk = X[:nb]
    Xm = np.concatenate(([0.0 + 0.0j], X[: nb - 1]))
    raw = Xk.real**2 + Xk.imag**2
    dif = Xk - Xm
    return np.maximum(raw, 0.5 * (dif.real**2 + dif.imag**2))


def interbin_power_oversampled(X):
    """SURVEY 8(f) row f4, reading G12b: the 2x-oversampled ("Fourier interpolated") spectrum of
    N = 2 Nb half bins,
        P'_{2k}   = |X_k|^2,
        P'_{2k+1} = (pi/4)^2 |X_k - X_{k+1}|^2,      k = 0..Nb-1,
    with X_0 <- 0 first (G13) and X_Nb the Nyquist bin of the FFT.  (pi/4)(X_k - X_{k+1}) is the
    two-bin estimate of the Fourier amplitude at k + 1/2 of Ransom et al. 2002, the paper's reference
    for scalloping: a tone midway between two bins, which the raw bins see at
    (2/pi)^2 = 0.405 of its power, comes back at 1.0.  Half bin q is the frequency q / (2 T_obs)."""
    X = np.array(X, dtype=np.complex128)
    nb = X.size - 1
    X[0] = 0.0
    out = np.empty(2 * nb, dtype=np.float64)
    out[0::2] = X[:nb].real**2 + X[:nb].imag**2
    dif = X[:nb] - X[1:nb + 1]
    out[1::2] = (math.pi / 4.0) ** 2 * (dif.real**2 + dif.imag**2)
    return out


def block_medians(P, window):
    """m_b = median(P[bW:(b+1)W]) (mean of the two middle order statistics), reading G15 of
    "Fourier de-reddening"."""
    P = np.asarray(P, dtype=np.float64)
    assert P.size % window == 0
    return np.median(P.reshape(-1, window), axis=1)


def median_baseline(m_b, n_bins, window):
    """m(k): linear interpolation of the block medians between block centres
    c_b = bW + (W-1)/2, constant beyond the first/last centre (G15)."""
    centres = np.arange(m_b.size, dtype=np.float64) * window + (window - 1) / 2.0
    return np.interp(np.arange(n_bins, dtype=np.float64), centres, m_b)


def normalise(P, m_b, window):
    """P^_k = P_k ln2 / m(k) (median of a unit-mean exponential is ln2: PAPER.md:L77 chi^2_2);
    P^_0 = 0 (G13); bins whose baseline is not positive are set to 0."""
    P = np.asarray(P, dtype=np.float64)
    m = median_baseline(np.asarray(m_b, dtype=np.float64), P.size, window)
    out = np.zeros_like(P)
    ok = m > 0
    out[ok] = P[ok] * LN2 / m[ok]
    out[0] = 0.0
    return out


# ----------------------------------------------------------------------------------------------
# O7  harmonic sum
# ----------------------------------------------------------------------------------------------
def harmonic_sums(p_hat, folds: Iterable[int] = (0, 1, 2, 3, 4)):
    """S_L[k] = sum_{m=1}^{2^L} P^[ floor((k m + 2^(L-1)) / 2^L) ]  (eq 9, equal
    weights L73; index reading G16: bin k of fold L is the bin of the highest summed harmonic,
    lower harmonics are taken at the nearest bin, halves rounded up).  Returns {L: float64[Nb]}."""
    p_hat = np.asarray(p_hat, dtype=np.float64)
    k = np.arange(p_hat.size, dtype=np.int64)
    out = {}
    for L in folds:
        n = 1 << L
        half = n >> 1
        S = np.zeros_like(p_hat)
        for m in range(1, n + 1):
            S += p_hat[(k * m + half) >> L]
        out[int(L)] = S
    return out


# ----------------------------------------------------------------------------------------------
# O8/O9  significance and candidates
# ----------------------------------------------------------------------------------------------
def sigma_constants(fold: int):
    """(mu_n, s_n) of sqrt(S) for S ~ Gamma(n, 1), n = 2^L summed unit-mean exponentials
    (PAPER.md:L77): mu_n = Gamma(n + 1/2)/Gamma(n), s_n = sqrt(n - mu_n^2).  At n = 1 these are
    the printed constants sqrt(pi/4), sqrt(1 - pi/4) of eq 11; reading G17."""
    n = 1 << int(fold)
    mu = math.exp(math.lgamma(n + 0.5) - math.lgamma(n))
    return mu, math.sqrt(n - mu * mu)


def sigma_of_power(S, fold: int):
    """sigma_L = (sqrt(S_L) - mu_n)/s_n  (eq 11 L83 generalised, G17)."""
    mu, s = sigma_constants(fold)
    return (np.sqrt(np.asarray(S, dtype=np.float64)) - mu) / s


def sigma_to_power(fold: int, sigma: float) -> float:
    """Inverse map: the summed power at which sigma_L equals ``sigma``."""
    mu, s = sigma_constants(fold)
    return (mu + sigma * s) ** 2


def lowest_bin_oversampled(n_samples, tsamp, f_min):
    """k_lo in half bins (G12b): twice lowest_bin's, so that both modes cut at the same frequency."""
    return 2 * lowest_bin(n_samples, tsamp, f_min)


def lowest_bin(n_samples, tsamp, f_min):
    """k_lo = ceil(f_min * N * tsamp) (G20)."""
    return int(math.ceil(f_min * (float(n_samples) * float(tsamp))))


def candidates_from_sums(sums, template_id, sigma_threshold, k_lo):
    """{(template, L, k, S, sigma)}: sigma_L[k] >= sigma_thr and k >= k_lo * 2^L (reading G19 of
    "peak detection": plain threshold, no merging).  Sorted by (L, k)."""
    out = []
    for L in sorted(sums):
        S = sums[L]
        sig = sigma_of_power(S, L)
        k = np.nonzero(sig >= sigma_threshold)[0]
        k = k[k >= (k_lo << L)]
        out.extend((int(template_id), int(L), int(kk), float(S[kk]), float(sig[kk])) for kk in k)
    return out


# ----------------------------------------------------------------------------------------------
# whole path for one template / a bank
# ----------------------------------------------------------------------------------------------
def spectrum_of_template(series, tsamp, tmpl, window=1024, fill=None, idx=None, oversample=False):
    """Steps O1-O6 for one template.  ``idx`` overrides the computed source indices (used by the
    parity tests to re-run the oracle with an excused tie flipped).  ``oversample``: the 2x-oversampled
    spectrum of reading G12b (N half bins instead of N/2 bins).  Returns a dict."""
    x = np.asarray(series, dtype=np.float32)
    if fill is None:
        fill = fill_value(x)
    if idx is None:
        idx = resample_indices(x.size, tsamp, tmpl)
    y = gather(x, idx, fill)
    P = interbin_power_oversampled(rfft_forward(y)) if oversample else interbin_power(rfft_forward(y))
    m_b = block_medians(P, window)
    return {"idx": idx, "resampled": y, "power": P, "medians": m_b, "normalised": normalise(P, m_b, window)}


def search_template(series, tsamp, tmpl, template_id=0, folds=(0, 1, 2, 3, 4), sigma_threshold=6.0,
                    window=1024, f_min=0.1, fill=None, idx=None, oversample=False):
    """Steps O1-O9 for one template: list of (template, L, k, S, sigma); with ``oversample`` k counts
    half bins (fundamental frequency k / (2^(L+1) T_obs))."""
    spec = spectrum_of_template(series, tsamp, tmpl, window, fill, idx, oversample)
    sums = harmonic_sums(spec["normalised"], folds)
    k_lo = (lowest_bin_oversampled if oversample else lowest_bin)(len(series), tsamp, f_min)
    return candidates_from_sums(sums, template_id, sigma_threshold, k_lo)


def search(series, tsamp, templates: Sequence, first_template_id=0, folds=(0, 1, 2, 3, 4),
           sigma_threshold=6.0, window=1024, f_min=0.1, fill=None):
    """The path of PAPER.md Alg. 1 (L677-707) + L660 for every template of a bank, one after the
    other.  Returns the candidate list sorted by (template, L, k)."""
    x = np.asarray(series, dtype=np.float32)
    if fill is None:
        fill = fill_value(x)
    out = []
    for i, tmpl in enumerate(np.asarray(templates, dtype=np.float64).reshape(-1, 5)):
        out.extend(search_template(x, tsamp, tmpl, first_template_id + i, folds, sigma_threshold,
                                   window, f_min, fill))
    return out


# ----------------------------------------------------------------------------------------------
# f2  front-end whitening once per series ("Fourier birdie
#     zapping, ..., Fourier de-reddening", L660 "Fourier de-reddenning").  The paper names the steps
#     and gives no formulas: reading G25 of DESIGN.md section 3 -- PARITY UNPINNED BY THE PAPER,
#     pinned by closed forms in tests/test_oracle_pins.py (a series that is already white is
#     returned unchanged up to the estimator's 1/sqrt(W) scatter; a red series comes out flat; a
#     zapped tone disappears; kappa normalises white noise to the same level as the per-template
#     estimator of G15).
# ----------------------------------------------------------------------------------------------
def whiten_series(series, window=1024, zap_bins=()):
    """x -> x': X = rfft(x); P_k = |X_k|^2 (raw, no interbinning); m(k) = the G15 baseline of P
    (block medians of `window` bins, linear interpolation between block centres); X'_k =
    X_k / sqrt(m(k) / ln2) for 1 <= k < N/2, X'_0 = X'_{N/2} = 0, and X'_k = 0 for every k in a
    zapped range [lo, hi) ("birdie zap"); x' = irfft(X') * sqrt(N): for noise E|X'_k|^2 = 1, so by
    Parseval sum_j x'_j^2 = N, i.e. unit variance.  Returns x' as float32."""
    x = np.asarray(series, dtype=np.float32).astype(np.float64)
    n = x.size
    X = np.fft.rfft(x)
    nb = n // 2
    P = X[:nb].real ** 2 + X[:nb].imag ** 2
    m = median_baseline(block_medians(P, window), nb, window)
    Xw = np.zeros_like(X)
    ok = m > 0
    ok[0] = False
    Xw[:nb][ok] = X[:nb][ok] / np.sqrt(m[ok] / LN2)
    for lo, hi in zap_bins:
        Xw[int(lo):int(hi)] = 0.0
    return (np.fft.irfft(Xw, n) * math.sqrt(float(n))).astype(np.float32)


def whitened_level(series_white, window=1024, zap_bins=()):
    """kappa: the ONE normalisation constant of a whitened series, replacing the per-template block
    medians of O6: kappa = ln2 / mean_b(m_b), m_b = block medians of the interbinned spectrum of
    the un-resampled whitened series.  P^_k = kappa * P_k for every template.
    Blocks touched by a zapped range are left out of the mean (reading G25): a range [lo, hi) zeroes
    X'_lo..X'_{hi-1}, which lowers the interbinned powers P_lo..P_hi and with them the medians of the blocks
    lo // W .. hi // W -- to 0 once half a block is zapped -- and kappa would grow by about 1 / (1 - zapped
    fraction of the band), raising every sigma.  If every block is touched, all blocks are used."""
    P = interbin_power(rfft_forward(series_white))
    m_b = block_medians(P, window)
    keep = np.ones(m_b.size, dtype=bool)
    for lo, hi in zap_bins:
        keep[int(lo) // window: int(hi) // window + 1] = False
    if not keep.any():
        keep[:] = True
    return LN2 / float(np.mean(m_b[keep]))


def spectrum_of_template_whitened(series_white, kappa, tsamp, tmpl, fill=None, idx=None):
    """Steps O1-O5, interbinning, and the constant normalisation P^ = kappa P (P^_0 = 0)."""
    x = np.asarray(series_white, dtype=np.float32)
    if fill is None:
        fill = fill_value(x)
    if idx is None:
        idx = resample_indices(x.size, tsamp, tmpl)
    y = gather(x, idx, fill)
    P = interbin_power(rfft_forward(y))
    Ph = kappa * P
    Ph[0] = 0.0
    return {"idx": idx, "resampled": y, "power": P, "normalised": Ph}


def search_template_whitened(series_white, kappa, tsamp, tmpl, template_id=0, folds=(0, 1, 2, 3, 4), sigma_threshold=6.0,
                             f_min=0.1, fill=None, idx=None):
    spec = spectrum_of_template_whitened(series_white, kappa, tsamp, tmpl, fill, idx)
    sums = harmonic_sums(spec["normalised"], folds)
    return candidates_from_sums(sums, template_id, sigma_threshold, lowest_bin(len(series_white), tsamp, f_min))
