"""Pins for the CPU oracle (oracle/tb_oracle.py): what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible slip in the
oracle (dropped term, wrong sign or index, transposed operand) fails at least one of them.
Citations are PAPER.md line numbers; T-numbers are SURVEY.md §4 / DESIGN.md §5.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import tb_oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ T1 / T3 / T11: index map
def test_t1_tau_zero_is_identity():
    n = 4096
    for tmpl in [(60.0, 0.0, 1.0, 0.0, 0.0), (33.0, 0.0, 2.5, 0.3, 1.1)]:
        idx = orc.resample_indices(n, 1e-3, tmpl)
        assert np.array_equal(idx, np.arange(n))


def test_t3_first_index_is_zero():
    rng = np.random.default_rng(3)
    for _ in range(20):
        tmpl = (rng.uniform(5, 90), rng.uniform(0, 4), rng.uniform(0, 2 * np.pi),
                rng.uniform(0, 0.5), rng.uniform(0, 2 * np.pi))
        assert orc.resample_indices(1024, 1e-3, tmpl)[0] == 0
        circ = (tmpl[0], tmpl[1], tmpl[2], 0.0, 0.0)
        assert orc.resample_indices(1024, 1e-3, circ)[0] == 0


def test_t11_monotone_and_out_of_range_bound():
    rng = np.random.default_rng(11)
    n, tsamp = 1 << 16, 64e-6
    T = n * tsamp
    for _ in range(8):
        p = rng.uniform(0.1 * T, 0.35 * T)
        tau = rng.uniform(0.01, 0.8) * p / (2 * np.pi)      # orbital speed v/c = tau*Omega in [0.01, 0.8]
        e, om, a = rng.uniform(0, 0.1), rng.uniform(0, 2 * np.pi), rng.uniform(0, 2 * np.pi)
        stretch = tau * 2 * np.pi / p * math.sqrt((1 + e) / (1 - e))
        assert stretch < 1
        idx = orc.resample_indices(n, tsamp, (p, tau, a, e, om))
        assert np.all(np.diff(idx) >= 0), "gather map must be monotone when tau*Omega*sqrt((1+e)/(1-e)) < 1"
        max_shift = np.max(np.abs(np.arange(n) - idx))
        assert max_shift <= 2 * tau * (1 + e) / tsamp + 1          # |delta| <= 2 tau (1+e)/tsamp
        oob = np.count_nonzero((idx < 0) | (idx >= n))
        assert oob <= 2 * (max_shift + 1)


def test_shift_sign_and_magnitude_closed_form():
    """Circular quarter-orbit: delta(P/4) - delta(0) = tau (sin(pi/2+phi0) - sin(phi0)) / tsamp
    (eq A1 at e=0, L666; eq 4).  phi0 = 0 -> +tau/tsamp: source index j - tau/tsamp."""
    tsamp, p, tau = 1e-3, 4.096, 0.25
    idx = orc.resample_indices(2048, tsamp, (p, tau, 0.0, 0.0, 0.0))
    j = 1024                                   # t = P/4
    assert idx[j] == j - 250
    j = 2047                                   # just before t = P/2: delta -> ~0+
    assert abs((j - idx[j])) <= 1


# ------------------------------------------------------------------ T2: e = 0 reduces to circular
def test_t2_kepler_path_at_e0_is_the_circular_closed_form():
    n, tsamp = 1 << 15, 1e-3
    tmpl = (47.0, 0.8, 1.3, 0.0, 0.0)
    j = np.arange(n)
    a = orc.roemer_delay(j, tsamp, tmpl)                       # closed form
    b = orc.roemer_delay(j, tsamp, tmpl, force_kepler=True)    # Newton path, e = 0, omega = 0
    assert np.array_equal(a, b)                                # Newton returns E = M exactly
    assert np.array_equal(orc.resample_indices(n, tsamp, tmpl),
                          orc.resample_indices(n, tsamp, tmpl, force_kepler=True))
    # omega != 0 at e = 0: tau sin(M + omega)  (A1 with E = M)
    om = 0.7
    c = orc.roemer_delay(j, tsamp, (47.0, 0.8, 1.3, 0.0, om))
    d = orc.roemer_delay(j, tsamp, (47.0, 0.8, 1.3 + om, 0.0, 0.0))
    assert np.max(np.abs(c - d)) < 1e-14


# ------------------------------------------------------------------ T4: Kepler solve
def _load_series():
    C, S = {}, {}
    with open(os.path.join(GOLDEN, "appendix_b_series.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            kind, k, pw, num, den = line.split()
            (C if kind == "C" else S).setdefault(int(k), []).append((int(pw), Fraction(int(num), int(den))))
    return C, S


def test_t4_kepler_residual_and_appendix_b_series():
    C, S = _load_series()
    M = np.linspace(0.0, 2 * np.pi, 20001)
    for e in (0.01, 0.05, 0.08, 0.1):
        E = orc.kepler_solve(M, e)
        assert np.max(np.abs(E - e * np.sin(E) - M)) <= 1e-12
        cosE = sum(sum(float(c) * e**p for p, c in terms) * np.cos(k * M) for k, terms in C.items())
        sinE = sum(sum(float(c) * e**p for p, c in terms) * np.sin(k * M) for k, terms in S.items())
        # the printed series is truncated after e^6: remainder O(e^7) (measured ~1.16 e^7)
        assert np.max(np.abs(np.cos(E) - cosE)) < 2.0 * e**7 + 1e-15
        assert np.max(np.abs(math.sqrt(1 - e * e) * np.sin(E) - sinE)) < 2.0 * e**7 + 1e-15


def test_kepler_against_bisection_high_eccentricity():
    for e in (0.3, 0.7, 0.9):
        for M in (0.1, 1.0, 2.5, 3.5, 6.0):
            lo, hi = M - 1.0, M + 1.0
            for _ in range(200):
                mid = 0.5 * (lo + hi)
                if mid - e * math.sin(mid) < M:
                    lo = mid
                else:
                    hi = mid
            assert abs(float(orc.kepler_solve(np.array([M]), e)[0]) - 0.5 * (lo + hi)) < 1e-12


# ------------------------------------------------------------------ gather
def test_gather_and_fill():
    x = np.arange(8, dtype=np.float32) * 10
    idx = np.array([0, 0, 2, 7, 8, -1, 3, 100])
    y = orc.gather(x, idx, np.float32(-5))
    assert y.dtype == np.float32
    assert y.tolist() == [0, 0, 20, 70, -5, -5, 30, -5]
    assert orc.fill_value(np.array([1, 2, 3, 6], dtype=np.float32)) == np.float32(3.0)


# ------------------------------------------------------------------ T5 / T6: FFT
def test_t5_parseval():
    y = np.random.default_rng(5).standard_normal(1 << 14).astype(np.float32)
    X = orc.rfft_forward(y)
    n = y.size
    lhs = np.sum(y.astype(np.float64) ** 2)
    rhs = (abs(X[0]) ** 2 + 2 * np.sum(np.abs(X[1:-1]) ** 2) + abs(X[-1]) ** 2) / n
    assert abs(lhs - rhs) < 1e-9 * lhs


def test_t6_bruteforce_dft_1024():
    n = 1024
    y = np.random.default_rng(6).standard_normal(n).astype(np.float32)
    jk = np.outer(np.arange(n // 2 + 1), np.arange(n))
    brute = (np.exp(-2j * np.pi * jk / n) * y.astype(np.float64)).sum(axis=1)
    assert np.max(np.abs(orc.rfft_forward(y) - brute)) < 1e-9


# ------------------------------------------------------------------ T7: interbinning closed forms
def test_t7_interbin_integer_and_half_bin_tone():
    n, k0, A = 1 << 16, 1 << 13, 0.5
    j = np.arange(n)
    ref = (A * n / 2) ** 2
    P = orc.interbin_power(orc.rfft_forward(A * np.cos(2 * np.pi * k0 * j / n)))
    assert P.size == n // 2
    assert abs(P[k0] / ref - 1) < 1e-9
    assert abs(P[k0 + 1] / ref - 0.5) < 1e-9          # 1/2 |0 - X_k0|^2
    assert P[k0 - 1] / ref < 1e-12
    P = orc.interbin_power(orc.rfft_forward(A * np.cos(2 * np.pi * (k0 + 0.5) * j / n)))
    assert abs(P[k0] / ref - (2 / np.pi) ** 2) < 2e-3          # raw scalloped bin: 0.405
    assert abs(P[k0 + 1] / ref - 8 / np.pi**2) < 2e-3          # interbin recovers 0.811


def test_dc_is_removed_before_interbinning():
    y = np.ones(4096) * 7.0 + np.random.default_rng(1).standard_normal(4096)
    P = orc.interbin_power(orc.rfft_forward(y))
    assert P[0] == 0.0
    X = orc.rfft_forward(y)
    assert abs(P[1] - abs(X[1]) ** 2) < 1e-9 * abs(X[1]) ** 2   # no DC leakage through the difference term


# ------------------------------------------------------------------ medians / T8
def test_block_median_by_hand():
    P = np.array([5, 1, 4, 2, 8, 7, 3, 6, 10, 10, 10, 10, 0, 0, 0, 1], dtype=float)
    assert orc.block_medians(P, 8).tolist() == [4.5, 5.5]        # (4+5)/2 ; sorted 0,0,0,1,10,10,10,10 -> (1+10)/2


def test_baseline_interpolation_by_hand():
    m = orc.median_baseline(np.array([2.0, 4.0]), 8, 4)          # centres 1.5 and 5.5
    assert np.allclose(m, [2, 2, 2.25, 2.75, 3.25, 3.75, 4, 4])


def test_t8_exponential_noise_normalises_to_unit_mean():
    P = np.random.default_rng(8).exponential(3.7, 1 << 18)
    mb = orc.block_medians(P, 1024)
    assert abs(np.mean(mb) / 3.7 - math.log(2)) < 0.01           # median = ln2 * mean (L77)
    ph = orc.normalise(P, mb, 1024)
    assert ph[0] == 0.0
    assert abs(np.mean(ph[1:]) - 1.0) < 0.01


def test_normalise_where_the_baseline_is_not_positive():
    """"ours" (G15): a bin whose interpolated median is <= 0 normalises to 0, not to inf or NaN.  Blocks 1 and 2
    are all zero, so m(k) = 0 between their centres; towards blocks 0 and 3 the baseline is interpolated and
    positive, and the ordinary formula applies there (values by hand)."""
    W = 4
    P = np.array([2, 2, 2, 2, 0, 0, 0, 0, 0, 0, 0, 0, 6, 6, 6, 6], dtype=np.float64)
    mb = orc.block_medians(P, W)
    assert mb.tolist() == [2.0, 0.0, 0.0, 6.0]
    out = orc.normalise(P, mb, W)
    assert np.all(np.isfinite(out)) and out[0] == 0.0
    assert np.all(out[4:12] == 0.0)                                  # numerator 0 or baseline 0: both give 0
    assert out[1] == pytest.approx(2 * math.log(2) / 2.0)            # k = 1 < centre 1.5: flat baseline m = 2
    assert out[3] == pytest.approx(2 * math.log(2) / (2.0 * (1 - 1.5 / 4)))      # k = 3: m = 2 (1 - (3 - 1.5)/4)
    assert out[15] == pytest.approx(math.log(2))                     # flat beyond the last centre: m = 6
    Pz = np.zeros(16)
    assert np.all(orc.normalise(Pz + 1.0, np.zeros(4), W) == 0.0)    # a positive power over a zero baseline -> 0


# ------------------------------------------------------------------ harmonic sums
def _round_half_up(fr: Fraction) -> int:
    return math.floor(fr + Fraction(1, 2))


def test_t6_harmonic_sum_bruteforce_from_eq9():
    nb = 512
    p = np.random.default_rng(9).exponential(1.0, nb)
    sums = orc.harmonic_sums(p)
    for L in range(5):
        n = 1 << L
        for k in range(nb):
            s = sum(p[_round_half_up(Fraction(k * m, n))] for m in range(1, n + 1))   # eq 9
            assert abs(sums[L][k] - s) < 1e-12


def test_harmonic_comb():
    nb, k0, Pk = 4096, 100, 3.0
    p = np.zeros(nb)
    p[[k0 * m for m in range(1, 17)]] = Pk
    sums = orc.harmonic_sums(p)
    for L in range(5):
        assert sums[L][k0 << L] == Pk * (1 << L)                 # all 2^L harmonics collected
        assert np.argmax(sums[L]) == (k0 << L) or L < 4
    assert sums[0][k0] == Pk


def test_harmonic_nesting_identity():
    p = np.random.default_rng(10).exponential(1.0, 2048)
    s = orc.harmonic_sums(p)
    k = np.arange(2048)
    for L in range(1, 5):
        odd = sum(p[(k * m + (1 << (L - 1))) >> L] for m in range(1, (1 << L) + 1, 2))
        assert np.allclose(s[L], s[L - 1] + odd, rtol=0, atol=1e-12)


# ------------------------------------------------------------------ T9: significance
def _golden_eq11():
    vals, ex = {}, []
    with open(os.path.join(GOLDEN, "eq11_constants.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            a, b, *c = line.split()
            if a == "example":
                ex.append((int(b), float(c[0])))
            else:
                vals[a] = float(b)
    return vals, ex


def test_t9_sigma_map_is_eq11_at_one_harmonic():
    vals, ex = _golden_eq11()
    mu, s = orc.sigma_constants(0)
    assert abs(mu - vals["sqrt_pi_over_4"]) < 1e-12
    assert abs(s - vals["sqrt_1_minus_pi_over_4"]) < 1e-12
    for n_trials, snr in ex:
        assert abs(float(orc.sigma_of_power(math.log(n_trials), 0)) - snr) < 5e-5
    for L in range(5):
        assert abs(float(orc.sigma_of_power(orc.sigma_to_power(L, 6.0), L)) - 6.0) < 1e-12


def test_sigma_constants_against_monte_carlo():
    rng = np.random.default_rng(17)
    for L in range(5):
        n = 1 << L
        r = np.sqrt(rng.gamma(n, 1.0, 2_000_000))
        mu, s = orc.sigma_constants(L)
        assert abs(r.mean() - mu) < 2e-3
        assert abs(r.std() - s) < 2e-3


def test_lowest_bin_and_candidate_rule():
    assert orc.lowest_bin(1 << 17, 1e-3, 0.1) == 14               # ceil(13.1072)
    sums = {1: np.array([0.0] * 40)}
    thr = orc.sigma_to_power(1, 6.0)
    sums[1][27] = thr * 1.0001      # below k_lo * 2^L = 28: rejected
    sums[1][28] = thr * 1.0001      # accepted
    sums[1][30] = thr * 0.9999      # below threshold
    c = orc.candidates_from_sums(sums, 5, 6.0, 14)
    assert [(t, L, k) for t, L, k, _, _ in c] == [(5, 1, 28)]


# ------------------------------------------------------------------ T10: end to end on C1
def test_t10_injected_pulsar_found_with_true_template(c1):
    x, tsamp = c1.series, c1.tsamp
    cands = orc.search_template(x, tsamp, c1.templates[0], 0)
    assert len(cands) > 0
    best = max(cands, key=lambda c: c[4])
    f_spin = 1.0 / c1.pulsars[0][0]
    L, k = best[1], best[2]
    assert L == 3                                   # only 10 harmonics of 50 Hz fit below Nyquist
    assert abs(k / ((1 << L) * c1.t_obs) - f_spin) < 1.0 / c1.t_obs
    assert best[4] > 12.0
    # every fold peaks at the spin frequency (fold 4 at the 25 Hz alias of the 8-harmonic sum)
    for fold, expect in ((0, 6554), (1, 13107), (2, 26214), (3, 52429)):
        b = max((c for c in cands if c[1] == fold), key=lambda c: c[4])
        assert abs(b[2] - expect) <= 1
    # a wrong template and the un-resampled series do not find it
    for tmpl in (c1.templates[5], (60.0, 0.0, 0.0, 0.0, 0.0), (60.0, 0.5, 1.0 + np.pi, 0.0, 0.0)):
        assert orc.search_template(x, tsamp, tmpl, 1) == []


def test_tie_distance_arbiter():
    d = orc.tie_distance(np.array([0, 10, 100]), 1e-3, (60.0, 0.0, 0.0, 0.0, 0.0))
    assert np.allclose(d, 0.5)                       # delta = 0 everywhere: as far from a tie as possible
    d64 = orc.shift_in_samples(np.arange(5000), 1e-3, (60.0, 0.5, 1.0, 0.0, 0.0))
    dl = orc.tie_distance(np.arange(5000), 1e-3, (60.0, 0.5, 1.0, 0.0, 0.0))
    assert np.max(np.abs(np.abs((d64 - np.floor(d64)) - 0.5) - dl)) < 1e-9


# ------------------------------------------------------------------ eq A1 at e > 0: the assembly of roemer_delay
def test_roemer_delay_elliptical_against_the_printed_series():
    """Delta = tau[(sum_k C_k cos kM - e) sin(omega) + (sum_k S_k sin kM) cos(omega)]: eq A1
    with cos E and sqrt(1-e^2) sin E replaced by the PRINTED e-series (eqs 15-16, App. B
    L719-747; the S-series already carries the sqrt(1-e^2) factor).  Truncated after e^6, so the
    two agree to ~1.2 e^7 per unit tau; a dropped sqrt(1-e^2), a swapped sin/cos(omega) or a
    missing -e moves the delay by >= e^2/2 tau."""
    C, S = _load_series()
    tsamp, p_orb, tau, phi0 = 1e-3, 37.0, 2.5, 0.4
    j = np.arange(0, 40000, 7)
    M = 2 * np.pi / p_orb * (j * tsamp) + phi0
    for e in (0.01, 0.05, 0.1):
        cosE = sum(sum(float(c) * e**p for p, c in terms) * np.cos(k * M) for k, terms in C.items())
        qsinE = sum(sum(float(c) * e**p for p, c in terms) * np.sin(k * M) for k, terms in S.items())
        for om in (0.3, 1.2, 4.0):
            series = tau * ((cosE - e) * math.sin(om) + qsinE * math.cos(om))
            got = orc.roemer_delay(j, tsamp, (p_orb, tau, phi0, e, om))
            assert np.max(np.abs(got - series)) < (2.0 * e**7 * (abs(math.sin(om)) + abs(math.cos(om))) + 1e-14) * tau


def test_roemer_delay_elliptical_closed_form_points():
    """Points of eq A1 where Kepler's equation (eq 3) solves by hand:
    M = 0 -> E = 0; M = pi -> E = pi; M = pi/2 - e -> E = pi/2."""
    tau, tsamp = 3.0, 1e-3
    j0 = np.zeros(1, dtype=np.int64)
    for e in (0.05, 0.3, 0.7):
        q = math.sqrt(1 - e * e)
        for om in (0.3, 1.2, 4.0):
            d = orc.roemer_delay(j0, tsamp, (50.0, tau, 0.0, e, om))[0]
            assert abs(d - tau * (1 - e) * math.sin(om)) < 1e-14 * tau
            d = orc.roemer_delay(j0, tsamp, (50.0, tau, math.pi, e, om))[0]
            assert abs(d + tau * (1 + e) * math.sin(om)) < 1e-14 * tau
            d = orc.roemer_delay(j0, tsamp, (50.0, tau, math.pi / 2 - e, e, om))[0]
            assert abs(d - tau * (-e * math.sin(om) + q * math.cos(om))) < 1e-14 * tau
            # a quarter of a period later in TIME (not at j = 0): t = P/4, phi0 = pi/2 - e - pi/2
            p = 40.96
            d = orc.roemer_delay(np.array([10240]), tsamp, (p, tau, -e, e, om))[0]
            assert abs(d - tau * (-e * math.sin(om) + q * math.cos(om))) < 1e-12 * tau


# ------------------------------------------------------------------ G10: the extended-precision tie decision
def _exact_shift(j, tsamp, tmpl, digits=50):
    """delta_j of eqs 3 / A1 / Alg. 1 L682-702 evaluated with mpmath at `digits` decimal digits on
    the exact values of the double-precision inputs (independent of the oracle: own formulas)."""
    import mpmath as mp
    with mp.workdps(digits):
        p_orb, tau, phi0, e, om = (mp.mpf(float(v)) for v in tmpl)
        ts = mp.mpf(float(tsamp))

        def delay(t):
            M = 2 * mp.pi / p_orb * t + phi0
            E = mp.findroot(lambda x: x - e * mp.sin(x) - M, M) if e != 0 else M
            return tau * ((mp.cos(E) - e) * mp.sin(om) + mp.sqrt(1 - e * e) * mp.sin(E) * mp.cos(om))

        return (delay(mp.mpf(int(j)) * ts) - delay(mp.mpf(0))) / ts


def _tau_for_shift(j, tsamp, tmpl_unit_tau, target):
    """tau (double) for which delta_j = target, from the exact shift per unit tau."""
    import mpmath as mp
    with mp.workdps(50):
        return float(mp.mpf(target) / _exact_shift(j, tsamp, tmpl_unit_tau))


@pytest.mark.parametrize("p_orb,phi0,e,om,j,n_int,off", [
    (60.0, 1.0, 0.0, 0.0, 20011, 250, 3e-8),         # circular, moderate: fp64 would also get this right
    (60.0, 1.0, 0.0, 0.0, 20011, 250, 2e-10),        # inside the north_star tie window's decade
    (55.0, 2.2, 0.08, 1.2, 31337, 400, 3e-8),        # elliptical
    (107.3, 0.7, 0.0, 0.0, 8000011, -60000, 2e-9),   # C4-like extreme (tau/tsamp ~ 5e4, j ~ 2^23)
    # 2e-11 from the tie: plain fp64 (phase error ~1e-10 samples here) decides these WRONGLY on one
    # side; only the extended-precision re-decision gets both sides right
    (107.3, 0.7, 0.0, 0.0, 8001020, -60000, 2e-11),
    (95.1, 2.9, 0.07, 2.2, 8000011, 110000, 2e-11),
    (95.1, 2.9, 0.07, 2.2, 8001020, 110000, 2e-11),
])
def test_tie_branch_decides_like_the_exact_formula(p_orb, phi0, e, om, j, n_int, off):
    """A sample constructed to sit `off` below / above a rounding tie (delta_j = n + 1/2 -+ off):
    resample_indices must take floor(delta + 1/2) of the EXACT delta (50-digit mpmath), i.e. the
    re-decision of lines "near" in resample_indices is what fixes the integer (reading G10)."""
    import mpmath as mp
    tsamp = 64e-6 if j > 1000000 else 1e-3
    for side in (-1, +1):
        tau = _tau_for_shift(j, tsamp, (p_orb, 1.0, phi0, e, om), mp.mpf(n_int) + mp.mpf(1) / 2 + side * mp.mpf(off))
        tmpl = (p_orb, tau, phi0, e, om)
        exact = _exact_shift(j, tsamp, tmpl)
        with mp.workdps(50):
            frac_off = float(exact - mp.floor(exact) - mp.mpf(1) / 2)
            want = int(j) - int(mp.floor(exact + mp.mpf(1) / 2))
        assert 0.3 * off < abs(frac_off) < 1.7 * off and np.sign(frac_off) == side     # the construction holds (tau is rounded to a double)
        assert want == int(j) - (n_int + (1 if side > 0 else 0))
        # the oracle's own fp64 shift is inside TIE_GUARD, so the extended-precision branch decides
        d64 = orc.shift_in_samples(np.array([j]), tsamp, tmpl)[0]
        assert abs((d64 - math.floor(d64)) - 0.5) < orc.TIE_GUARD
        n = j + 1
        idx = orc.resample_indices(n, tsamp, tmpl)
        assert idx[j] == want
        assert abs(orc.tie_distance(np.array([j]), tsamp, tmpl)[0] - abs(frac_off)) < 0.1 * off


# ------------------------------------------------------------------ G2-G4: the sign convention against eq A2 taken literally
def test_sign_convention_against_literal_eq_a2():
    """Eq A2 read literally, with NO inverse-map construction: the pulsar-frame
    time of the sample observed at t is t' = t - Delta_R(t).  Alg. 1 L702 gathers S[j - Delta_j/tsamp]
    (reading G3), which is the map t = t' - Delta_R(t'), i.e. the opposite sign (G4: the paper is
    at odds with itself: eq 2/4 vs A2 vs Alg. 1).  A sign flip of Delta_R is phi0 -> phi0 + pi for
    a circular orbit, and the two maps then differ only by the second-order term
    tau^2 Omega cos(.) sin(.) (0.4 ms here, against a 1 ms pulse).  So a series synthesised from
    literal A2 must be found by the oracle with the template at phi0 + pi and NOT at phi0."""
    n, tsamp, p_spin, p_orb, tau, phi0 = 1 << 16, 1e-3, 0.020, 40.0, 0.05, 0.9
    rng = np.random.default_rng(4242)
    t = np.arange(n) * tsamp
    t_psr = t - tau * np.sin(2 * np.pi / p_orb * t + phi0)             # eq A2 with eq A1 at e = 0
    ph = t_psr / p_spin
    d = ph - np.rint(ph)
    sig = 0.05 / (2.0 * math.sqrt(2.0 * math.log(2.0)))
    x = (rng.standard_normal(n) + 0.45 * np.exp(-0.5 * (d / sig) ** 2)).astype(np.float32)
    found = orc.search_template(x, tsamp, (p_orb, tau, phi0 + np.pi, 0.0, 0.0), 0)
    assert found, "literal-A2 signal not recovered at phi0 + pi"
    best = max(found, key=lambda c: c[4])
    assert abs(best[2] / ((1 << best[1]) * n * tsamp) - 1.0 / p_spin) < 1.0 / (n * tsamp)
    assert best[4] > 10.0
    assert orc.search_template(x, tsamp, (p_orb, tau, phi0, 0.0, 0.0), 0) == []
    assert orc.search_template(x, tsamp, (p_orb, 0.0, phi0, 0.0, 0.0), 0) == []      # and not without resampling


# ------------------------------------------------------------------ f2: whitening once per series (reading G25)
def test_whitening_closed_form_impulse():
    """x = delta at j0: |X_k|^2 = 1 for every k, so every block median is 1 and X'_k = sqrt(ln2) X_k for
    0 < k < N/2, X'_0 = X'_{N/2} = 0:  x'_j = sqrt(N ln2) (delta_{j j0} - 1/N - (-1)^(j-j0)/N)."""
    n, j0 = 4096, 777
    x = np.zeros(n, dtype=np.float32)
    x[j0] = 1.0
    got = orc.whiten_series(x, window=256).astype(np.float64)
    j = np.arange(n)
    want = math.sqrt(n * math.log(2)) * ((j == j0).astype(float) - 1.0 / n - (-1.0) ** (j - j0) / n)
    assert np.max(np.abs(got - want)) < 1e-5


def test_whitening_flattens_red_noise_and_keeps_white_noise():
    rng = np.random.default_rng(25)
    n = 1 << 16
    w = rng.standard_normal(n)
    xw = orc.whiten_series((3.0 * w + 10.0).astype(np.float32))        # white, scaled, with a DC offset
    assert abs(xw.std() - 1.0) < 0.01 and abs(xw.mean()) < 1e-6
    assert np.corrcoef(xw, w)[0, 1] > 0.995                             # only the estimator's scatter is added
    assert np.max(np.abs(orc.whiten_series((7.0 * (3.0 * w + 10.0)).astype(np.float32)) - xw)) < 1e-4   # scale-free
    red = np.cumsum(w) * 0.05 + w                                       # random walk + white: power ~ 1/f^2 at low f
    band = lambda y, a, b: np.mean(np.abs(np.fft.rfft(y))[a:b] ** 2)
    assert band(red, 16, 512) / band(red, n // 4, n // 2) > 20.0
    xr = orc.whiten_series(red.astype(np.float32))
    # where the spectrum is steep the piecewise-linear baseline of 1024-bin medians lags by a few per cent
    assert abs(band(xr, 1024, 4096) / band(xr, n // 4, n // 2) - 1.0) < 0.15
    assert abs(band(xr, 8192, 16384) / band(xr, n // 4, n // 2) - 1.0) < 0.05
    assert abs(band(xr, 1024, n // 2) / n - 1.0) < 0.02                 # E|X'_k|^2 = N for a unit-variance series


def test_whitening_zaps_birdies():
    rng = np.random.default_rng(26)
    n, k0 = 1 << 14, 3000
    x = (rng.standard_normal(n) + 0.5 * np.cos(2 * np.pi * k0 * np.arange(n) / n)).astype(np.float32)
    kept = np.abs(np.fft.rfft(orc.whiten_series(x)))
    zapped = np.abs(np.fft.rfft(orc.whiten_series(x, zap_bins=[(k0 - 1, k0 + 2)])))
    assert kept[k0] > 20 * np.median(kept)                              # a block median does not remove a tone
    assert np.all(zapped[k0 - 1:k0 + 2] < 1e-3) and zapped[k0 + 5] > 1.0


def test_whitened_level_matches_the_per_template_normalisation():
    """kappa P of a whitened white series has the same level as P ln2 / m(k) (G15) of the raw one."""
    rng = np.random.default_rng(27)
    x = rng.standard_normal(1 << 17).astype(np.float32)
    tmpl = (60.0, 0.3, 1.0, 0.0, 0.0)
    a = orc.spectrum_of_template(x, 1e-3, tmpl)["normalised"]
    xw = orc.whiten_series(x)
    b = orc.spectrum_of_template_whitened(xw, orc.whitened_level(xw), 1e-3, tmpl)["normalised"]
    assert b[0] == 0.0 and abs(np.mean(b[1:]) / np.mean(a[1:]) - 1.0) < 0.01
    assert abs(np.median(b[1:]) - math.log(2)) < 0.01                   # kappa puts the median at ln2, like G15


def test_t10_on_the_whitened_series(c1):
    xw = orc.whiten_series(c1.series)
    kappa = orc.whitened_level(xw)
    cands = orc.search_template_whitened(xw, kappa, c1.tsamp, c1.templates[0], 0)
    best = max(cands, key=lambda c: c[4])
    assert (best[1], best[2]) == (3, 52429) and best[4] > 12.0
    assert orc.search_template_whitened(xw, kappa, c1.tsamp, c1.templates[5], 1) == []


def test_whitened_level_ignores_zapped_blocks():
    """A birdie list covering 6 % of the band (reading G25): the normalised powers of the UNzapped bins of a
    whitened white series must still average 1 (median ln 2).  With the zapped blocks inside the mean of the
    block medians, kappa -- and every normalised power -- comes out 1 / (1 - 0.06) too large."""
    rng = np.random.default_rng(31)
    n, W = 1 << 17, 1024
    x = rng.standard_normal(n).astype(np.float32)
    zap = [(8 * W, 10 * W), (30 * W + 100, 31 * W + 900), (50 * W, 50 * W + 300)]           # whole blocks, a straddle, a part
    xw = orc.whiten_series(x, W, zap)
    P = orc.interbin_power(orc.rfft_forward(xw))
    clear = np.ones(n // 2, dtype=bool)
    clear[0] = False
    for lo, hi in zap:
        clear[lo - 1: hi + 2] = False
    kappa = orc.whitened_level(xw, W, zap)
    assert abs(np.median(kappa * P[clear]) - math.log(2)) < 0.012
    level_all = orc.whitened_level(xw, W)                                  # the round-2 rule: every block
    touched = {b for lo, hi in zap for b in range(lo // W, hi // W + 1)}
    assert touched == {8, 9, 10, 30, 31, 50}
    assert level_all / kappa > 1.04                                        # what the zapped blocks would have cost
    # no zap ranges: unchanged; every block zapped: falls back to all blocks instead of dividing by nothing
    assert orc.whitened_level(xw, W, ()) == level_all
    assert np.isfinite(orc.whitened_level(xw, W, [(0, n // 2)]))


# ------------------------------------------------------------------ f4: the ELL7 approximate-orbit delay (reading G26)
def test_ell_table_is_the_printed_appendix_b():
    """The oracle's coefficient table against the numbers typed independently into the golden file
    from PAPER.md:L719-747."""
    C, S = _load_series()
    assert {k: sorted((pw, fr.numerator, fr.denominator) for pw, fr in v) for k, v in C.items()} == \
           {k: sorted(tuple(t) for t in v) for k, v in orc.ELL_C.items()}
    assert {k: sorted((pw, fr.numerator, fr.denominator) for pw, fr in v) for k, v in S.items()} == \
           {k: sorted(tuple(t) for t in v) for k, v in orc.ELL_S.items()}


def test_ell_delay_against_the_kepler_solve_and_closed_forms():
    tsamp, p_orb, tau, phi0 = 1e-3, 41.0, 3.0, 0.9
    j = np.arange(0, 60000, 11)
    for e in (0.0, 0.02, 0.1):
        for om in (0.0, 0.7, 2.9, 5.1):
            tm = (p_orb, tau, phi0, e, om)
            ell = orc.roemer_delay(j, tsamp, tm, model="ell")
            bt = orc.roemer_delay(j, tsamp, tm, force_kepler=True)
            assert np.max(np.abs(ell - bt)) < (2.0 * e**7 * (abs(math.sin(om)) + abs(math.cos(om))) + 2e-15) * tau
    # e = 0: C_1 = S_1 = 1, everything else 0: tau sin(M + omega) exactly (eq A1 at e = 0)
    M = 2 * np.pi / p_orb * (j * tsamp) + phi0
    assert np.max(np.abs(orc.roemer_delay(j, tsamp, (p_orb, tau, phi0, 0.0, 1.3), model="ell") - tau * np.sin(M + 1.3))) < 1e-14 * tau
    # first order in e by hand: cos E = cos M + e (cos 2M - 1)/2 + O(e^2), sqrt(1-e^2) sin E = sin M + e sin 2M / 2 + O(e^2)
    e = 1e-4
    d = orc.roemer_delay(j, tsamp, (p_orb, tau, phi0, e, 0.4), model="ell")
    first = tau * ((np.cos(M) + e * (np.cos(2 * M) - 1) / 2 - e) * math.sin(0.4) + (np.sin(M) + e * np.sin(2 * M) / 2) * math.cos(0.4))
    assert np.max(np.abs(d - first)) < 2.0 * e * e * tau
    # and the index map: identical to BT's except where the 1.2 e^7 tau / tsamp difference crosses a rounding tie
    tm = (p_orb, 0.5, phi0, 0.05, 0.7)
    a = orc.resample_indices(1 << 15, tsamp, tm, model="ell")
    b = orc.resample_indices(1 << 15, tsamp, tm)
    assert a[0] == 0 and np.count_nonzero(a != b) <= 2 and np.max(np.abs(a - b)) <= 1
    tm = (400.0, 20.0, phi0, 0.3, 0.7)                      # e = 0.3: the truncation, 1.2 e^7 tau / tsamp = 5 samples, is visible
    a = orc.resample_indices(1 << 18, tsamp, tm, model="ell")
    b = orc.resample_indices(1 << 18, tsamp, tm)
    assert np.count_nonzero(a != b) > 1000 and 2 <= np.max(np.abs(a - b)) <= 8


# ------------------------------------------------------------------ G12b: 2x-oversampled interbinning
def test_oversampled_interbinning_closed_forms():
    """Tone at an integer bin: P'_{2k0} = (A N / 2)^2 and both neighbouring half bins (pi/4)^2 of it; tone
    midway between bins: the raw bins see (2/pi)^2 = 0.405, the half bin between them 1.0 (N -> infinity);
    even entries are the raw powers; X_0 is removed before differencing; the last half bin uses the Nyquist bin."""
    n, A = 4096, 0.7
    j = np.arange(n)
    full = (A * n / 2) ** 2
    X = orc.rfft_forward(A * np.cos(2 * np.pi * 200 * j / n + 0.4) + 5.0)            # + DC
    P = orc.interbin_power_oversampled(X)
    assert P.size == n and P[0] == 0.0
    assert P[400] == pytest.approx(full, rel=1e-12)
    assert P[399] == pytest.approx((math.pi / 4) ** 2 * full, rel=1e-9) and P[401] == pytest.approx((math.pi / 4) ** 2 * full, rel=1e-9)
    assert P[1] == pytest.approx((math.pi / 4) ** 2 * abs(X[1]) ** 2, rel=1e-12, abs=1e-18)      # DC did not leak in
    raw = np.abs(X[: n // 2]) ** 2
    raw[0] = 0.0
    assert np.allclose(P[0::2], raw, rtol=1e-13, atol=1e-12)
    Xh = orc.rfft_forward(A * np.cos(2 * np.pi * 200.5 * j / n + 0.4))
    Ph = orc.interbin_power_oversampled(Xh)
    assert Ph[400] / full == pytest.approx((2 / math.pi) ** 2, rel=5e-3) and Ph[402] / full == pytest.approx((2 / math.pi) ** 2, rel=5e-3)
    assert Ph[401] / full == pytest.approx(1.0, rel=5e-3)
    assert np.argmax(Ph) == 401
    Xn = orc.rfft_forward(np.cos(np.pi * j))                                          # Nyquist tone
    assert orc.interbin_power_oversampled(Xn)[-1] == pytest.approx((math.pi / 4) ** 2 * n * n, rel=1e-12)
    # white noise: even half bins have unit mean (in units of N sigma^2), odd ones pi^2/8
    rng = np.random.default_rng(4)
    Pn = orc.interbin_power_oversampled(orc.rfft_forward(rng.standard_normal(1 << 16))) / (1 << 16)
    assert Pn[0::2].mean() == pytest.approx(1.0, rel=0.02) and Pn[1::2].mean() == pytest.approx(math.pi ** 2 / 8, rel=0.02)


def test_oversampled_search_recovers_a_half_bin_pulsar():
    """End to end on a scalloped signal: a sinusoid midway between two bins in noise.  The oversampled
    search finds it in the odd half bin with ~pi^2/4 more power than the plain spectrum's raw bins; its
    candidate frequencies are k / (2^(L+1) T_obs); k_lo doubles."""
    n, tsamp = 1 << 14, 1e-3
    rng = np.random.default_rng(8)
    j = np.arange(n)
    x = (rng.standard_normal(n) + 0.12 * np.cos(2 * np.pi * 1000.5 * j / n)).astype(np.float32)
    tmpl = (50.0, 0.0, 0.0, 0.0, 0.0)                                                 # tau = 0: no resampling
    over = orc.search_template(x, tsamp, tmpl, 0, (0,), 5.0, window=1024, oversample=True)
    assert orc.lowest_bin_oversampled(n, tsamp, 0.1) == 2 * orc.lowest_bin(n, tsamp, 0.1)
    best = max(over, key=lambda c: c[4])
    assert best[2] == 2001                                                            # half bin 2 * 1000.5
    spec = orc.spectrum_of_template(x, tsamp, tmpl, 1024, oversample=True)
    plain = orc.spectrum_of_template(x, tsamp, tmpl, 1024)
    assert spec["power"].size == n and spec["medians"].size == n // 1024 and plain["power"].size == n // 2
    raw_best = max(spec["power"][2000], spec["power"][2002])                          # even half bins are the raw |X_k|^2
    assert spec["power"][2001] > 1.8 * raw_best                                       # (pi/2)^2 = 2.47 without noise
    assert plain["power"][1001] == pytest.approx(0.5 * (4 / math.pi) ** 2 * spec["power"][2001], rel=1e-12)   # G12's 1/2 |dX|^2
