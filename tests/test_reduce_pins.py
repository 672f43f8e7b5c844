"""Pins for the candidate-reduction oracle (oracle/tb_reduce.py).

The paper names the step and gives no algorithm (reading G24), so the pins are hand-built
detection lists whose groups are worked out by hand below, plus the C1 end-to-end case.  None of
these tests touches the CUDA path.
"""
import numpy as np

from oracle import tb_oracle as orc
from oracle import tb_reduce as red


def D(t, L, k, sigma, power=None):
    return (t, L, k, float(power if power is not None else sigma * sigma), float(sigma))


def test_r1_runs_of_adjacent_bins_become_one_peak():
    dets = [D(0, 2, 10, 5), D(0, 2, 11, 7), D(0, 2, 12, 6),      # one run, best = bin 11
            D(0, 2, 14, 9),                                       # gap of two bins: a peak of its own
            D(0, 3, 11, 8),                                       # same bin, other fold: separate
            D(1, 2, 13, 4)]                                       # other template: does not bridge 12..14
    peaks, srt, owner = red.peaks_from_detections(dets[::-1])     # input order is irrelevant
    assert [(p[0], p[1], p[2], p[5]) for p in peaks] == [(0, 2, 11, 3), (0, 2, 14, 1), (0, 3, 11, 1), (1, 2, 13, 1)]
    assert owner == [0, 0, 0, 1, 2, 3]
    # equal sigma inside a run: the lowest bin wins
    peaks, _, _ = red.peaks_from_detections([D(0, 0, 5, 6), D(0, 0, 6, 6)])
    assert peaks[0][2] == 5 and peaks[0][5] == 2


def test_frequency_is_exact_in_sixteenths_of_a_bin():
    assert red.freq16(3, 52429) == 104858           # 6553.625 * 16
    assert red.freq16(4, 52429) == 52429            # 3276.8125 * 16
    assert red.freq16(0, 6554) == 104864


def test_r3_relation_by_hand():
    Fh = red.freq16(3, 52429)                       # 104858 (6553.625 bins)
    # second harmonic seen in fold 0 at bin 13107: |1 * 209712 - 2 * 104858| = 4 <= 16
    assert red.related(Fh, red.freq16(0, 13107))
    # two bins further: 209744 - 209716 = 28 > 16, and no other p/q <= 16 comes closer than 28
    assert not red.related(Fh, red.freq16(0, 13109))
    # the 1/7 sub-harmonic alias in fold 4, bin 14981 (936.3125): |7 * 14981 - 1 * 104858| = 9
    assert red.related(Fh, red.freq16(4, 14981))
    # 5/3: fold 2 bin 43690 (10922.5): |3 * 174760 - 5 * 104858| = 10
    assert red.related(Fh, red.freq16(2, 43690))
    # the relation is symmetric (swap p and q)
    assert red.related(red.freq16(0, 13107), Fh)
    # a ratio that needs p = 17 is out: F_b = 17 F_h, and 17/1 has no equivalent with p, q <= 16
    assert not red.related(16 * 1000, 16 * 17000)
    assert red.related(16 * 1000, 16 * 16000)
    # tolerance is in fundamental bins: 1000 vs 1001.0 bins related (16/16), 1001.5 not (24/16), q = p = 1 ... 16
    assert red.related(16000, 16016) and not red.related(16000, 16024)
    assert red.related(16000, 16024, tol16=24)


def test_r3_greedy_heads_only_absorb():
    """A (1000 bins, 10 sigma), B = 3/2 A (8 sigma), C = 13/16 B = 1218.75 bins (6 sigma).
    C/A = 39/32 is not within a bin of any p/q with p, q <= 16 (nearest: 11/9 A = 1222.2, 6/5 A =
    1200), so A absorbs B only; B is absorbed and absorbs nothing; C heads its own group."""
    A, B, C = D(0, 0, 1000, 10), D(0, 0, 1500, 8), D(0, 2, 4875, 6)          # 4875 / 4 = 1218.75
    groups, member_of = red.reduce_candidates([C, B, A])
    assert [(g["bin"], g["fold"], g["n_peaks"]) for g in groups] == [(1000, 0, 2), (4875, 2, 1)]
    assert member_of == [0, 0, 1]                                             # sorted input order: A, B, C
    # had C been the strongest, it would absorb B (16 * 1218.75 = 13 * 1500) and A would stand alone
    groups, _ = red.reduce_candidates([D(0, 2, 4875, 12), B, A])
    assert [(g["bin"], g["n_peaks"]) for g in groups] == [(4875, 2), (1000, 1)]


def test_r3_across_templates_and_r4_counts():
    dets = [D(3, 3, 8000, 9), D(3, 3, 8001, 8.5),      # template 3: one peak of two detections at 1000.0 bins
            D(7, 3, 8001, 7),                          # template 7 sees the same frequency (1000.125)
            D(7, 0, 2000, 6.5),                        # ... and its second harmonic in fold 0
            D(5, 1, 1234 * 2 + 1, 8),                  # an unrelated signal at 1234.5 bins, template 5
            D(9, 1, 1234 * 2 + 1, 8)]                  # the same in template 9 with EQUAL sigma: template 5 heads
    groups, member_of = red.reduce_candidates(dets)
    assert len(groups) == 2
    g0, g1 = groups
    assert (g0["template"], g0["fold"], g0["bin"], g0["n_peaks"], g0["n_detections"], g0["n_templates"]) == (3, 3, 8000, 3, 4, 2)
    assert (g1["template"], g1["fold"], g1["bin"], g1["n_peaks"], g1["n_detections"], g1["n_templates"]) == (5, 1, 2469, 2, 2, 2)
    # sorted detections: (3,3,8000) (3,3,8001) (5,1,2469) (7,0,2000) (7,3,8001) (9,1,2469)
    assert member_of == [0, 0, 1, 0, 0, 1]


def test_sigma_is_ranked_as_float32():
    """Two heads whose sigmas differ only beyond float32: the tie falls back to (template, fold, bin)."""
    a, b = D(2, 0, 1000, 7.000000001), D(1, 0, 1307, 7.0)        # 1.307 is no p/q with p, q <= 16
    groups, _ = red.reduce_candidates([a, b])
    assert [g["template"] for g in groups] == [1, 2]


def test_empty_and_single():
    assert red.reduce_candidates([]) == ([], [])
    groups, member_of = red.reduce_candidates([D(4, 4, 99, 6)])
    assert len(groups) == 1 and member_of == [0] and groups[0]["n_detections"] == 1


def test_c1_reduces_to_one_group_at_50_hz(c1):
    """the 76 raw detections of C1's true template are one 20 ms pulsar."""
    dets = orc.search_template(c1.series, c1.tsamp, c1.templates[0], 0)
    assert len(dets) == 76
    groups, member_of = red.reduce_candidates(dets)
    assert len(groups) == 1 and set(member_of) == {0}
    g = groups[0]
    assert (g["fold"], g["bin"], g["n_detections"]) == (3, 52429, 76)
    assert abs(g["bin"] / (8 * c1.t_obs) - 50.0) < 1.0 / c1.t_obs


def test_two_unrelated_signals_stay_apart():
    """20 ms (fundamental 6553.6 bins) and 31.7 ms (4134.76 bins): ratio 1.585, more than a bin away
    from every p/q <= 16 at these frequencies (nearest 19/12 needs p = 19; 8/5 f2 = 6615.6)."""
    f1, f2 = 6553.6, 4134.76
    dets = []
    for L in range(5):
        dets += [D(0, L, int(round(f1 * 2**L)), 9 + L), D(0, L, int(round(f2 * 2**L)), 8 + L)]
    dets += [D(0, 0, int(round(2 * f1)), 6.5), D(0, 0, int(round(3 * f2)), 6.2)]
    groups, _ = red.reduce_candidates(dets)
    assert len(groups) == 2
    assert [g["n_peaks"] for g in groups] == [6, 6]
    assert {round(g["bin"] / 2 ** g["fold"]) for g in groups} == {6554, 4135}


def test_vectorised_relation_equals_the_double_loop():
    rng = np.random.default_rng(5)
    Fh = int(rng.integers(500, 200000))
    Fb = rng.integers(100, 400000, 3000)
    Fb[:200] = (Fh * rng.integers(1, 17, 200)) // rng.integers(1, 17, 200) + rng.integers(-20, 21, 200)   # near-harmonic cases
    want = np.array([red.related(Fh, int(f)) for f in Fb])
    assert want.sum() > 50 and (~want).sum() > 50
    assert np.array_equal(red.related_many(Fh, Fb), want)
