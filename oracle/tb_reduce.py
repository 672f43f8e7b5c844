"""CPU oracle for the candidate reduction step.

TEST INFRASTRUCTURE ONLY (same rules as oracle/tb_oracle.py: only tests/, smoke() and bench.py's
cpu_baseline / --impl reference legs may import it; it shares no code with the CUDA path).

PAPER.md:L660 (App. A): the pipeline "additionally runs a candidate reduction algorithm by
grouping together multiple detections of the same candidate".  The paper gives no algorithm, so
everything below is reading G24 of DESIGN.md section 3 -- PARITY UNPINNED BY THE PAPER; the pins
in tests/test_reduce_pins.py fix it against hand-built lists, exact rational arithmetic and the
C1 end-to-end case (76 raw detections of one 50 Hz pulsar -> one group).

Reading G24, in the order it is applied to the raw detection list {(template, fold L, bin k, S, sigma)}:

  R1  peaks.  Within one (template, fold) a maximal run of detections in ADJACENT bins
      (k, k+1, k+2, ...) is one spectral peak (interbinning, G12, puts a tone into two
      neighbouring bins; a smeared signal into a few more).  The peak is the run's detection of
      highest sigma (ties: the lowest bin).  Its frequency, in bins of the fundamental (units of
      1/T_obs), is f = k / 2^L (G16: bin k of fold L indexes the highest of the 2^L harmonics);
      here it is kept as the exact integer F = k * 2^(4-L) = 16 f.
  R2  order.  Peaks are ranked by (sigma descending, template, fold, bin ascending).  sigma is
      compared as the float32 value the search produced (so that both sides rank identically).
  R3  distillation (greedy, as in PEASOUP's harmonic / trial distillers that L660's pipeline is
      built on): walk the ranking; a peak not yet absorbed becomes the HEAD of a new group and
      absorbs every weaker, not yet absorbed peak -- of ANY template and fold -- that is
      harmonically related to it:
          related(h, b)  <=>  there are integers 1 <= p, q <= H with |q F_b - p F_h| <= tol16
      (H = 16 = the largest number of summed harmonics; tol16 = 16 * tolerance in fundamental
      bins, default 16 = one bin).  p/q = 1 joins the same frequency seen in other folds and in
      neighbouring templates; p/q != 1 joins harmonics and sub-harmonic aliases.
  R4  groups are numbered in head order; a group reports its head, the number of peaks and the
      number of raw detections it holds, and the number of distinct templates among them.
"""
from __future__ import annotations

import numpy as np

H_MAX = 16
TOL16_DEFAULT = 16


def peaks_from_detections(dets):
    """R1.  dets: iterable of (template, fold, bin, power, sigma).  Returns the list of peaks
    (template, fold, bin, power, sigma, n_detections, first_index) where first_index is the
    position of the run's first detection in the (template, fold, bin)-sorted list, plus that
    sorted list and, for each sorted detection, the index of its peak."""
    srt = sorted(dets, key=lambda d: (d[0], d[1], d[2]))
    peaks, owner = [], []
    i = 0
    while i < len(srt):
        j = i
        while j + 1 < len(srt) and srt[j + 1][0] == srt[i][0] and srt[j + 1][1] == srt[i][1] and srt[j + 1][2] == srt[j][2] + 1:
            j += 1
        run = srt[i:j + 1]
        best = run[0]
        for d in run[1:]:
            if np.float32(d[4]) > np.float32(best[4]):
                best = d
        peaks.append((best[0], best[1], best[2], best[3], best[4], len(run), i))
        owner.extend([len(peaks) - 1] * len(run))
        i = j + 1
    return peaks, srt, owner


def freq16(fold, k):
    """F = 16 f = k * 2^(4 - L): the peak's fundamental frequency in 1/16 bins, an exact integer."""
    return int(k) << (4 - int(fold))


def related(F_h, F_b, tol16=TOL16_DEFAULT, h_max=H_MAX):
    """R3's relation: min over 1 <= p, q <= H of |q F_b - p F_h| <= tol16 (plain double loop)."""
    for q in range(1, h_max + 1):
        for p in range(1, h_max + 1):
            if abs(q * F_b - p * F_h) <= tol16:
                return True
    return False


def related_many(F_h, F_b, tol16=TOL16_DEFAULT, h_max=H_MAX):
    """``related`` for an int64 array F_b at once (the same double loop, one array operation per (p, q))."""
    F_b = np.asarray(F_b, dtype=np.int64)
    out = np.zeros(F_b.shape, dtype=bool)
    for q in range(1, h_max + 1):
        for p in range(1, h_max + 1):
            out |= np.abs(q * F_b - p * int(F_h)) <= tol16
    return out


def reduce_candidates(dets, tol16=TOL16_DEFAULT, h_max=H_MAX):
    """R1-R4.  Returns (groups, member_of): groups = list of dicts in head order
    {template, fold, bin, power, sigma, n_peaks, n_detections, n_templates}; member_of[i] = group of
    the i-th detection of the (template, fold, bin)-sorted input."""
    peaks, srt, owner = peaks_from_detections(dets)
    rank = sorted(range(len(peaks)), key=lambda i: (-float(np.float32(peaks[i][4])), peaks[i][0], peaks[i][1], peaks[i][2]))
    F = np.array([freq16(peaks[i][1], peaks[i][2]) for i in rank], dtype=np.int64)      # in rank order
    group_of_rank = np.full(len(rank), -1, dtype=np.int64)
    groups = []
    for pos, h in enumerate(rank):
        if group_of_rank[pos] >= 0:
            continue
        g = len(groups)
        group_of_rank[pos] = g
        later = np.arange(pos + 1, len(rank))
        later = later[group_of_rank[later] < 0]
        absorbed = later[related_many(F[pos], F[later], tol16, h_max)] if later.size else later
        group_of_rank[absorbed] = g
        members = [h] + [rank[b] for b in absorbed]
        hp = peaks[h]
        groups.append({"template": hp[0], "fold": hp[1], "bin": hp[2], "power": hp[3], "sigma": hp[4],
                       "n_peaks": len(members), "n_detections": sum(peaks[m][5] for m in members),
                       "n_templates": len({peaks[m][0] for m in members})})
    group_of = [0] * len(peaks)
    for pos, i in enumerate(rank):
        group_of[i] = int(group_of_rank[pos])
    member_of = [group_of[o] for o in owner]
    return groups, member_of
