"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md §4).

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench, so it holds none
of the search method's arithmetic: it imports neither ``oracle/`` nor the CUDA binding.  What it
does contain is the *signal model* needed to synthesise a binary pulsar (eqs 1-6,
L666-672 eqs A1/A2) -- written here independently, for injection only.

The paper's own data (HTRU-S Lowlat, Terzan 5, PSR J0737-3039A, sigproc ``fake`` runs) are not
available; these series stand in for them by shape: length, sampling time, white Gaussian noise
 and orbital ranges.

Everything is numpy on the host; arrays are handed unchanged to the oracle and to the library.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

BASE_SEED = 211211991          # arXiv id 2112.11991
DUTY = 0.05                    # pulse FWHM / period
AMP_C1 = 0.3                   # BASELINE.json C1
N_C1 = 1 << 17


@dataclasses.dataclass
class Workload:
    name: str
    n_samples: int
    tsamp: float
    series: np.ndarray                 # float32[N]
    templates: np.ndarray              # float64[K,5] = (P_orb s, tau lt-s, phi0 rad, e, omega rad)
    true_ids: tuple                    # template ids holding an injected pulsar's parameters
    pulsars: tuple                     # ((P_spin, P_orb, tau, phi0, e, omega, amplitude), ...)
    folds: tuple = (0, 1, 2, 3, 4)
    sigma_threshold: float = 6.0
    median_window: int = 1024
    f_min: float = 0.1

    @property
    def t_obs(self) -> float:
        return self.n_samples * self.tsamp


# ------------------------------------------------------------------ signal model (injection only)
def _settle(step_fn, x, max_iter, tol):
    """x <- x - step_fn(x) up to max_iter times or until max|step| < tol.  When the last digit
    flickers between two values (x_k == x_{k-2}) the remaining iterations are skipped and the value
    the full loop would have ended on is returned, bit for bit: the tolerances below are tighter
    than one ulp of the larger arguments, so without this every call ran all max_iter iterations."""
    prev = None                                     # iterate before the last one
    for k in range(max_iter):
        step = step_fn(x)
        new = x - step
        if np.max(np.abs(step)) < tol:
            return new
        if prev is not None and np.array_equal(new, prev):          # period 2: new, x, new, x, ...
            return new if (max_iter - 1 - k) % 2 == 0 else x
        prev, x = x, new
    return x


def _ecc_anomaly(M, e):
    return _settle(lambda E: (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E)), M + e * np.sin(M), 60, 1e-15)


def _delay_and_rate(t, p_orb, tau, phi0, e, om):
    """Roemer delay (s) and its time derivative at pulsar-frame times t (eq A1)."""
    w = 2.0 * np.pi / p_orb
    E = _ecc_anomaly(w * t + phi0, e)
    sE, cE = np.sin(E), np.cos(E)
    q = math.sqrt(1.0 - e * e)
    d = tau * ((cE - e) * math.sin(om) + q * sE * math.cos(om))
    dd = tau * w * (-sE * math.sin(om) + q * cE * math.cos(om)) / (1.0 - e * cE)
    return d, dd


def emission_times(s, p_orb, tau, phi0, e, om):
    """Pulsar-frame time t' of the signal observed at s: solves s = t' - (Delta(t') - Delta(0))
    (eq A2 with the zero offset of L675), Newton in t'.  This is the exact inverse of the
    search's gather map (reading G3)."""
    d0, _ = _delay_and_rate(np.zeros(1), p_orb, tau, phi0, e, om)

    def step(t):
        d, dd = _delay_and_rate(t, p_orb, tau, phi0, e, om)
        return (t - (d - d0[0]) - s) / (1.0 - dd)

    return _settle(step, np.array(s, dtype=np.float64), 60, 1e-13)


def pulse_train(n, tsamp, p_spin, p_orb, tau, phi0, e, om, amp, duty=DUTY):
    """A * exp(-(d/sigma)^2/2), d = wrapped distance of frac(t'/P_spin) from 0,
    sigma = duty / (2 sqrt(2 ln 2)) (duty = FWHM / period)."""
    s = np.arange(n, dtype=np.float64) * tsamp
    ph = emission_times(s, p_orb, tau, phi0, e, om) / p_spin
    d = ph - np.rint(ph)
    sig = duty / (2.0 * math.sqrt(2.0 * math.log(2.0)))
    return amp * np.exp(-0.5 * (d / sig) ** 2)


def default_amplitude(n):
    """Same matched-filter S/N as C1's A = 0.3 at 2^17 samples (S/N^2 ~ A^2 * duty * N)."""
    return AMP_C1 * math.sqrt(N_C1 / n)


def _rng(config: int, extra: int = 0):
    return np.random.default_rng(BASE_SEED + (config - 1) + 1000 * extra)


def _bank(rng, k, p_lo, p_hi, t_lo, t_hi, elliptical=False, e_hi=0.1):
    """One rng.uniform call per parameter: all P_orb, all tau, all phi0 [, all e, all omega]."""
    p = rng.uniform(p_lo, p_hi, k)
    t = rng.uniform(t_lo, t_hi, k)
    a = rng.uniform(0.0, 2.0 * np.pi, k)
    if elliptical:
        e = rng.uniform(0.0, e_hi, k)
        o = rng.uniform(0.0, 2.0 * np.pi, k)
    else:
        e = np.zeros(k)
        o = np.zeros(k)
    return np.stack([p, t, a, e, o], axis=1)


# ------------------------------------------------------------------ the five configs
def config1(n_templates: int = 64) -> Workload:
    """C1 "PR1 ref": 2^17 @ 1 ms, N(0,1) + 20 ms pulsar (A=0.3, P_orb=60 s, tau=0.5, phi0=1);
    template 0 = truth, the rest P_orb~U[40,90] s, tau~U[0,1], phi0~U[0,2pi)."""
    n, tsamp = 1 << 17, 1e-3
    rng = _rng(1)
    noise = rng.standard_normal(n)
    psr = (0.020, 60.0, 0.5, 1.0, 0.0, 0.0, AMP_C1)
    bank = _bank(rng, n_templates - 1, 40.0, 90.0, 0.0, 1.0)
    templates = np.vstack([np.array([[60.0, 0.5, 1.0, 0.0, 0.0]]), bank])
    x = noise + pulse_train(n, tsamp, *psr)
    return Workload("C1", n, tsamp, x.astype(np.float32), templates, (0,), (psr,))


def config2(n_templates: int = 4096, log2n: int = 22) -> Workload:
    """C2: 2^22 @ 256 us, N(0,1) + 3 pulsars (P_spin~U[20,200] ms, P_orb~U[.1,.35]T,
    tau~U[.1,2]); templates 0-2 = truth, the rest drawn over the same ranges."""
    n, tsamp = 1 << log2n, 256e-6
    T = n * tsamp
    rng = _rng(2)
    noise = rng.standard_normal(n)
    ps = rng.uniform(0.020, 0.200, 3)
    po = rng.uniform(0.1 * T, 0.35 * T, 3)
    ta = rng.uniform(0.1, 2.0, 3)
    ph = rng.uniform(0.0, 2.0 * np.pi, 3)
    amp = default_amplitude(n)
    psrs = tuple((ps[i], po[i], ta[i], ph[i], 0.0, 0.0, amp) for i in range(3))
    bank = _bank(rng, max(n_templates - 3, 0), 0.1 * T, 0.35 * T, 0.1, 2.0)
    truth = np.array([[p[1], p[2], p[3], 0.0, 0.0] for p in psrs])
    x = noise
    for p in psrs:
        x = x + pulse_train(n, tsamp, *p)
    return Workload("C2", n, tsamp, x.astype(np.float32), np.vstack([truth, bank])[:max(n_templates, 3)],
                    (0, 1, 2), psrs)


def config3(n_templates: int = 16384, log2n: int = 25) -> Workload:
    """C3: 2^25 @ 128 us, 8-bit-quantised noise rescaled to float + 20 ms pulsar with
    P_orb=0.2T, tau=1.5; bank P_orb~U[.1,.33]T, tau~U[.05,3], phi0~U[0,2pi)."""
    n, tsamp = 1 << log2n, 128e-6
    T = n * tsamp
    rng = _rng(3)
    noise = rng.standard_normal(n)
    phi0 = rng.uniform(0.0, 2.0 * np.pi)
    psr = (0.020, 0.2 * T, 1.5, phi0, 0.0, 0.0, default_amplitude(n))
    bank = _bank(rng, n_templates - 1, 0.1 * T, 0.33 * T, 0.05, 3.0)
    v = noise + pulse_train(n, tsamp, *psr)
    q = np.clip(np.rint(32.0 * v) + 128.0, 0.0, 255.0)
    x = (q - 128.0) / 32.0
    templates = np.vstack([np.array([[psr[1], psr[2], psr[3], 0.0, 0.0]]), bank])
    return Workload("C3", n, tsamp, x.astype(np.float32), templates, (0,), (psr,))


def config4(n_templates: int = 8192, log2n: int = 23, tau_scale: float = 1.0) -> Workload:
    """C4: elliptical, 2^23 @ 64 us, N(0,1) + 25 ms pulsar (P_orb=0.15T, tau=4, e=0.08,
    omega=1.2); bank P_orb~U[.1,.2]T, tau~U[.5,8], phi0,omega~U[0,2pi), e~U[0,.1].
    ``tau_scale`` shrinks every tau for scaled-down test series (P_orb scales with T, so tau has
    to shrink too for the orbit to stay sub-luminal)."""
    n, tsamp = 1 << log2n, 64e-6
    T = n * tsamp
    rng = _rng(4)
    noise = rng.standard_normal(n)
    phi0 = rng.uniform(0.0, 2.0 * np.pi)
    psr = (0.025, 0.15 * T, 4.0 * tau_scale, phi0, 0.08, 1.2, default_amplitude(n))
    bank = _bank(rng, n_templates - 1, 0.1 * T, 0.2 * T, 0.5 * tau_scale, 8.0 * tau_scale, elliptical=True)
    x = noise + pulse_train(n, tsamp, *psr)
    templates = np.vstack([np.array([[psr[1], psr[2], psr[3], psr[4], psr[5]]]), bank])
    return Workload("C4", n, tsamp, x.astype(np.float32), templates, (0,), (psr,))


def config5(log2n: int = 23, n_circ: int = 256, n_ell: int = 256, noise: bool = True) -> Workload:
    """C5 throughput sweep: noise-only, tsamp = 64 us; 256 circular + 256 elliptical templates,
    P_orb~U[.1,.35]T, orbital speed v/c = tau*Omega~U[0.001,0.1], phi0,omega~U[0,2pi), e~U[0,.1].
    ``noise=False`` skips the (slow at 2^26) normal draw and returns a cheap uniform-bits series
    -- never used for parity, only for sizing runs."""
    n, tsamp = 1 << log2n, 64e-6
    T = n * tsamp
    rng = _rng(5, extra=log2n)
    x = rng.standard_normal(n, dtype=np.float32) if noise else rng.random(n, dtype=np.float32) - 0.5
    k = n_circ + n_ell
    p = rng.uniform(0.1 * T, 0.35 * T, k)
    beta = rng.uniform(0.001, 0.1, k)
    a = rng.uniform(0.0, 2.0 * np.pi, k)
    e = rng.uniform(0.0, 0.1, k)
    o = rng.uniform(0.0, 2.0 * np.pi, k)
    e[:n_circ] = 0.0
    o[:n_circ] = 0.0
    tau = beta * p / (2.0 * np.pi)
    templates = np.stack([p, tau, a, e, o], axis=1)
    return Workload(f"C5/2^{log2n}", n, tsamp, x, templates, (), ())


# ------------------------------------------------------------------ paper-shaped workloads
def config_paper(log2n: int = 24, n_templates: int = 1024) -> Workload:
    """The paper's own simulation set-up (Table 2): 2^24 samples at 256 us
    (72 min), a 15 ms pulsar in a P_orb = 8 h, e = 0.1 orbit around an 8 M_sun companion seen at 60 deg
    (tau = 6.6 lt-s), i.e. P_orb = 6.7 T_obs; bank: template 0 = truth, the rest P_orb~U[6,12] h,
    tau~U[0,7] lt-s, phi0, omega~U[0,2pi), e~U[0,0.1] (Table 1).  Duty cycle 10 % (Table 2)."""
    n, tsamp = 1 << log2n, 256e-6
    rng = _rng(6)
    noise = rng.standard_normal(n)
    phi0 = rng.uniform(0.0, 2.0 * np.pi)
    psr = (0.015, 8.0 * 3600.0, 6.6, phi0, 0.1, 1.0, default_amplitude(n) * math.sqrt(DUTY / 0.10))
    bank = _bank(rng, n_templates - 1, 6.0 * 3600.0, 12.0 * 3600.0, 0.0, 7.0, elliptical=True)
    x = noise + pulse_train(n, tsamp, *psr, duty=0.10)
    templates = np.vstack([np.array([[psr[1], psr[2], psr[3], psr[4], psr[5]]]), bank])
    return Workload("paper/2^%d" % log2n, n, tsamp, x.astype(np.float32), templates, (0,), (psr,))


def config_terzan(log2n: int = 28, n_templates: int = 8) -> Workload:
    """A Terzan-5-length series (7.2 h downsampled to 81.9 us = 2^28.2 samples): 2^28
    samples at 81.92 us (6.1 h), a 5 ms pulsar in a circular P_orb = 7 T_obs orbit, tau = 12 lt-s; bank:
    template 0 = truth, the rest P_orb~U[5,10] T_obs, tau~U[0,20] lt-s, phi0~U[0,2pi) ("a circular-orbit
    search between 5-10 T_obs ... up to a companion mass of 10 M_sun").  The series is built in float32
    chunks: at 2^28 samples every float64 temporary is 2 GiB."""
    n, tsamp = 1 << log2n, 81.92e-6
    T = n * tsamp
    rng = _rng(7)
    x = rng.standard_normal(n, dtype=np.float32)
    phi0 = rng.uniform(0.0, 2.0 * np.pi)
    psr = (0.005, 7.0 * T, 12.0, phi0, 0.0, 0.0, default_amplitude(n))
    bank = _bank(rng, n_templates - 1, 5.0 * T, 10.0 * T, 0.0, 20.0)
    step = 1 << 22
    sig = DUTY / (2.0 * math.sqrt(2.0 * math.log(2.0)))
    for j0 in range(0, n, step):
        s = (j0 + np.arange(min(step, n - j0), dtype=np.float64)) * tsamp
        ph = emission_times(s, *psr[1:6]) / psr[0]
        d = ph - np.rint(ph)
        x[j0:j0 + len(s)] += (psr[6] * np.exp(-0.5 * (d / sig) ** 2)).astype(np.float32)
    templates = np.vstack([np.array([[psr[1], psr[2], psr[3], 0.0, 0.0]]), bank])
    return Workload("terzan/2^%d" % log2n, n, tsamp, x, templates, (0,), (psr,))


def by_name(name: str, **kw) -> Workload:
    return {"C1": config1, "C2": config2, "C3": config3, "C4": config4, "C5": config5, "paper": config_paper, "terzan": config_terzan}[name](**kw)


def shard_templates(n_templates: int, rank: int, world: int):
    """Contiguous split of the template list over ranks (Alg. 1: templates are
    independent).  Returns (first, count); no rank exchanges anything with another."""
    base, rem = divmod(n_templates, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def synthetic_detections(seed: int, n_noise: int, n_signals: int = 3, n_templates: int = 8, nb: int = 1 << 16):
    """A seeded raw detection list for the candidate-reduction parity tests (no search arithmetic:
    just rows shaped like a search's output).  n_noise isolated rows at random (template, fold, bin)
    with sigma ~ 4 + Exp(0.5), plus n_signals "pulsars": a spin frequency seen in every fold of
    2-3 neighbouring templates as a run of 1-4 adjacent bins, with harmonics and sub-harmonic
    aliases, sigma up to ~20.  Rows are unique in (template, fold, bin); float32 sigma / power.
    Returns a structured array (template_id, fold, bin, power, sigma, pad) in random order."""
    rng = np.random.default_rng(BASE_SEED + 7000 + seed)
    rows = {}
    for _ in range(n_noise):
        key = (int(rng.integers(n_templates)), int(rng.integers(5)), int(rng.integers(16, nb)))
        rows[key] = 4.0 + rng.exponential(0.5)
    for s in range(n_signals):
        f = rng.uniform(200.0, nb / 40.0)                     # fundamental, bins
        peak = rng.uniform(9.0, 20.0)
        t0 = int(rng.integers(n_templates))
        for t in {t0, (t0 + 1) % n_templates, (t0 + int(rng.integers(3))) % n_templates}:
            for L in range(5):
                for num, den in ((1, 1), (2, 1), (3, 1), (1, 2), (1, 3), (3, 2), (5, 1)):
                    k = int(round(f * num / den * (1 << L)))
                    if not 16 <= k < nb - 8 or rng.random() < 0.25:
                        continue
                    for d in range(int(rng.integers(1, 5))):
                        rows[(t, L, k + d)] = max(4.0, peak * rng.uniform(0.4, 1.0) / (1.0 + 0.3 * abs(num - den)))
    dt = np.dtype([("template_id", "<u4"), ("fold", "<u4"), ("bin", "<u4"), ("power", "<f4"), ("sigma", "<f4"), ("pad", "<u4")])
    out = np.zeros(len(rows), dtype=dt)
    for i, ((t, L, k), sg) in enumerate(rows.items()):
        out[i] = (t, L, k, np.float32(sg * sg), np.float32(sg), 0)
    return out[rng.permutation(len(out))]
