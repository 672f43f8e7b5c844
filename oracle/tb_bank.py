"""CPU oracle for the random template-bank generator (PAPER.md sections 2.2-2.7).

TEST INFRASTRUCTURE ONLY (same rules as oracle/tb_oracle.py): only tests/ may import it, it shares
no code with the CUDA path, and every function cites the passage of /root/reference/PAPER.md it
follows.  Random numbers are INPUTS (arrays of uniforms in [0, 1)); nothing is drawn here.

What it computes, step by step in the paper's order:

  phase model ........ eq 1-2 (L35-41) with cos E and sqrt(1-e^2) sin E replaced by the printed
                       e-series of eqs 15-16 (L106-111, App. B); circular: eq 4 (L49)
  metric ............. g_ab = <d_a Phi d_b Phi>_T - <d_a Phi>_T <d_b Phi>_T        (eq 13)
                       <G>_T = (1/T) int_0^T G dt                                   (eq 14)
  projected metric ... gamma_ab = g_ab - g_fa g_fb / g_ff                           (eq 22)
  density ............ sqrt|det gamma|  ("distributed randomly with uniform probability based on
                       ... the square root of the determinant", L115; section 2.7)
  prior box .......... P_orb ~ U(P1, P2), tau ~ U(0, tau_max(Omega)) with eq 31 (L248),
                       alpha, psi ~ U(0, 2 pi), e ~ U(0, e_max)   (Table 1)
  placement .......... rejection sampling of  pdf ~ sqrt|gamma| x prior  (L263: "sample from a
                       probability density function that is proportional to sqrt|gamma| multiplied by
                       the prior"; the paper draws from it with an MCMC sampler, reading G28: plain
                       accept/reject with the caller's uniforms draws from the same pdf exactly)
  proper volume ...... V = int sqrt(gamma) d^n lambda (eq 17), Monte-Carlo over the proposals
  N_R ................ eq 20 (L131) and its expansion eq 21 (L136); C_n of eq 18 (L123)

Readings:
  G27  coordinates of the metric: Lambda = (f0, tau, Omega, alpha[, psi, e]) -- the parameters of eq 1-3
       as printed (L45-47); derivatives are those of eq 1-2 exactly (d/df includes the tau X term
       that eq 28's dimensionless form drops), so that eq 12's mismatch holds to O(Delta^3).
  G28  rejection sampling instead of emcee (above).
  G29  arithmetic: the time averages are Gauss-Legendre sums (exact to rounding for these band-
       limited integrands).  For P_orb >> T the metric is ill conditioned (cond 1e11 for typical
       points of the paper's box, 1e15 and more where e -> 0 makes psi and alpha degenerate), and
       the literal chain eq 13 -> eq 22 -> det loses cond * epsilon: fp64 is useless there and even
       x87 extended precision is off by 3e-5 typically and by a factor 4 at the degenerate points.
       So `density` evaluates the SAME formulas either in numpy.longdouble (fast; accurate to 1e-12
       for the several-orbit banks of BASELINE.json's configs, cond ~ 1e4) or, with digits=D, in
       D-digit mpmath arithmetic (density_mp), which is what the paper's box is compared in.

Against the paper's printed values (box of Table 1, eq 20 with eta = 0.9, m = 0.2):
  circular    paper 10 128      here N_R = 9946 +- 174 (20 000 proposals): reproduced, and pinned by
                                test_circular_template_count_of_the_papers_box
  elliptical  paper 2 047 716   here N_R ~ 60 (V = 2.5 +- 0.6): NOT reproduced.  Dropping the tau X term of
                                d Phi / d f (eq 28), the literal chain in float64 and the obvious omitted
                                Jacobians of eq 29 were tried: none gives the printed
                                count and the text does not say what was integrated.  The elliptical mode is
                                therefore PARITY UNPINNED against the paper; its pins below fix the mathematics
                                of reading G27, not the reading.

Parity pins (tests/test_bank_pins.py, -m "not gpu"):
  phase_derivatives ... every column against central finite differences of the EXACT phase (Kepler
                        solve of oracle/tb_oracle.py, no series) at e = 0.05
  metric .............. closed forms of the circular metric over whole orbits (g_tautau, g_alphaalpha,
                        g_taualpha, g_ftau, g_ff); eq 12: the mismatch 1 - |<exp(i dPhi)>|^2 computed
                        directly from the phase equals g_ab dL^a dL^b for small offsets along every
                        axis pair; quadrature converged (n vs 2n)
  projected metric .... min over a frequency offset of the direct mismatch = gamma_ab dl^a dl^b
  density ............. coordinate invariance: sqrt(det) transforms with the Jacobian under
                        (tau, psi) -> (X, Y) of eq 29
  tau_max ............. Kepler's third law in SI units by another route; the 6 h point by hand
  ball volume, N_R .... C_1 = 2, C_2 = pi, C_3 = 4 pi / 3; eq 20 inverts to the coverage; eq 21 is its limit
  rejection sampler ... brute force on a small proposal set; chi-square of the accepted histogram
                        against the density
"""
from __future__ import annotations

import math

import numpy as np

from oracle.tb_oracle import ELL_C, ELL_S

LD = np.longdouble
N_QUAD = 1024                       # Gauss-Legendre nodes of the time averages (G29); enough for ~100 orbital harmonics-cycles
T_SUN = 4.925490947e-6              # G M_sun / c^3 in seconds (IAU nominal solar mass parameter)


def _two_pi():
    return LD(8) * np.arctan(LD(1))


# ----------------------------------------------------------------------------------------------
# eq 15-16 / App. B: the e-series and their e-derivatives
# ----------------------------------------------------------------------------------------------
def ell_series(e):
    """C_k(e), k = 0..7 and S_k(e), k = 0..7 (S_0 = 0) with their derivatives dC_k/de, dS_k/de
    (PAPER.md:L106-111, L719-747), in longdouble."""
    e = LD(e)
    C = np.zeros(8, LD); S = np.zeros(8, LD); dC = np.zeros(8, LD); dS = np.zeros(8, LD)
    for k in range(8):
        for pw, num, den in ELL_C[k]:
            C[k] += LD(num) / LD(den) * e ** pw
            if pw > 0:
                dC[k] += LD(pw) * LD(num) / LD(den) * e ** (pw - 1)
    for k in range(1, 8):
        for pw, num, den in ELL_S[k]:
            S[k] += LD(num) / LD(den) * e ** pw
            if pw > 0:
                dS[k] += LD(pw) * LD(num) / LD(den) * e ** (pw - 1)
    return C, S, dC, dS


# ----------------------------------------------------------------------------------------------
# eq 1-4: the phase and its parameter derivatives
# ----------------------------------------------------------------------------------------------
def orbit_factor(t, lam, elliptical):
    """X(t) of Phi = 2 pi f0 [t + tau X(t)] and its derivatives with respect to M, psi and e.

    elliptical (eq 2 L41 with eqs 15-16):  X = sin(psi) sum_k C_k cos kM + cos(psi) sum_k S_k sin kM
    circular   (eq 4):                 X = sin M
    M = Omega t + alpha (eq 3).  lam = (tau, Omega, alpha[, psi, e]).  Returns X, X_M, X_psi, X_e.
    """
    t = np.asarray(t, LD)
    om, al = LD(lam[1]), LD(lam[2])
    M = om * t + al
    if not elliptical:
        return np.sin(M), np.cos(M), None, None
    psi, e = LD(lam[3]), LD(lam[4])
    C, S, dC, dS = ell_series(e)
    cc = sum(C[k] * np.cos(LD(k) * M) for k in range(8))             # cos E
    ss = sum(S[k] * np.sin(LD(k) * M) for k in range(1, 8))          # sqrt(1-e^2) sin E
    cc_M = sum(-LD(k) * C[k] * np.sin(LD(k) * M) for k in range(8))
    ss_M = sum(LD(k) * S[k] * np.cos(LD(k) * M) for k in range(1, 8))
    cc_e = sum(dC[k] * np.cos(LD(k) * M) for k in range(8))
    ss_e = sum(dS[k] * np.sin(LD(k) * M) for k in range(1, 8))
    sp, cp = np.sin(psi), np.cos(psi)
    return sp * cc + cp * ss, sp * cc_M + cp * ss_M, cp * cc - sp * ss, sp * cc_e + cp * ss_e


def phase(t, f0, lam, elliptical):
    """Phi(t; Lambda) of eq 1-2 (L35-41) / eq 4 (L49), series form (radians, longdouble)."""
    X = orbit_factor(t, lam, elliptical)[0]
    return _two_pi() * LD(f0) * (np.asarray(t, LD) + LD(lam[0]) * X)


def phase_derivatives(t, f0, lam, elliptical):
    """Rows d Phi / d(f0, tau, Omega, alpha[, psi, e]) at the times t (reading G27): shape [n_par, len(t)]."""
    t = np.asarray(t, LD)
    tau, f0 = LD(lam[0]), LD(f0)
    X, X_M, X_psi, X_e = orbit_factor(t, lam, elliptical)
    k = _two_pi()
    rows = [k * (t + tau * X), k * f0 * X, k * f0 * tau * t * X_M, k * f0 * tau * X_M]
    if elliptical:
        rows += [k * f0 * tau * X_psi, k * f0 * tau * X_e]
    return np.stack(rows)


# ----------------------------------------------------------------------------------------------
# eq 13, 14, 22: metric, projected metric, density
# ----------------------------------------------------------------------------------------------
_GL_CACHE = {}


def quadrature(t_obs, n_quad=N_QUAD):
    """Nodes in [0, T] and weights summing to 1: <G>_T = sum_i w_i G(t_i)  (eq 14).
    Gauss-Legendre: numpy's fp64 nodes refined to longdouble by Newton steps on P_n (with fp64 nodes
    the ill-conditioned metrics of G29 come out 50 times less accurate).  The rule is cached per
    n_quad (numpy's leggauss is an eigenvalue problem: slow when many worker processes call it)."""
    if n_quad not in _GL_CACHE:
        x = np.asarray(np.polynomial.legendre.leggauss(n_quad)[0], LD)

        def p_and_dp(x):
            p0, p1 = np.ones_like(x), x.copy()
            for k in range(2, n_quad + 1):
                p0, p1 = p1, ((2 * k - 1) * x * p1 - (k - 1) * p0) / LD(k)
            return p1, n_quad * (x * p1 - p0) / (x * x - 1)

        for _ in range(3):
            p, dp = p_and_dp(x)
            x = x - p / dp
        _GL_CACHE[n_quad] = (x, 2 / ((1 - x * x) * p_and_dp(x)[1] ** 2))
    x, w = _GL_CACHE[n_quad]
    return (LD(t_obs) / 2) * (x + 1), w / 2


def metric(f0, lam, t_obs, elliptical, n_quad=N_QUAD):
    """g_ab = <d_a Phi d_b Phi>_T - <d_a Phi>_T <d_b Phi>_T  (eq 13), index 0 = f0."""
    t, w = quadrature(t_obs, n_quad)
    D = phase_derivatives(t, f0, lam, elliptical)
    mean = D @ w
    return (D * w) @ D.T - np.outer(mean, mean)


def projected_metric(g):
    """gamma_ab = g_ab - g_fa g_fb / g_ff  (eq 22) on the orbital indices 1..n."""
    return g[1:, 1:] - np.outer(g[0, 1:], g[0, 1:]) / g[0, 0]


def determinant(a):
    """det of a small matrix by Gaussian elimination with partial pivoting, in the dtype of `a`
    (numpy.linalg has no longdouble path)."""
    a = np.array(a, dtype=LD)
    n = a.shape[0]
    det = LD(1)
    for c in range(n):
        p = c + int(np.argmax(np.abs(a[c:, c])))
        if a[p, c] == 0:
            return LD(0)
        if p != c:
            a[[c, p]] = a[[p, c]]
            det = -det
        det *= a[c, c]
        a[c + 1:, c:] -= np.outer(a[c + 1:, c] / a[c, c], a[c, c:])
    return det


def density(f0, lam, t_obs, elliptical, n_quad=N_QUAD, digits=None):
    """sqrt|det gamma| at lam = (tau, Omega, alpha[, psi, e])  (L115, L263).
    digits=None: longdouble (error ~ cond * 1e-19: fine for several-orbit banks, cond ~ 1e4);
    digits=D: the same formulas in D-digit mpmath arithmetic (density_mp), for the paper's own box
    where the condition number reaches 1e11..1e16 (psi and alpha degenerate as e -> 0)."""
    if digits:
        return density_mp(f0, lam, t_obs, elliptical, n_quad, digits)
    return float(np.sqrt(np.abs(determinant(projected_metric(metric(f0, lam, t_obs, elliptical, n_quad))))))


def density_mp(f0, lam, t_obs, elliptical, n_quad=N_QUAD, digits=50):
    """eq 13 -> eq 22 -> determinant, literally, in mpmath arithmetic of `digits` digits (reading G29).
    Time averages: composite Gauss-Legendre with mpmath's own 96-point rule on ceil(n_quad / 96) panels."""
    import mpmath as mp
    with mp.workdps(digits):
        tau, om, al = (mp.mpf(float(v)) for v in lam[:3])
        f0, t_obs = mp.mpf(float(f0)), mp.mpf(float(t_obs))
        k2 = 2 * mp.pi
        if elliptical:
            psi, e = mp.mpf(float(lam[3])), mp.mpf(float(lam[4]))
            C = [sum(mp.mpf(num) / den * e ** pw for pw, num, den in ELL_C[k]) for k in range(8)]
            S = [mp.mpf(0)] + [sum(mp.mpf(num) / den * e ** pw for pw, num, den in ELL_S[k]) for k in range(1, 8)]
            dC = [sum(pw * mp.mpf(num) / den * e ** (pw - 1) for pw, num, den in ELL_C[k] if pw) for k in range(8)]
            dS = [mp.mpf(0)] + [sum(pw * mp.mpf(num) / den * e ** (pw - 1) for pw, num, den in ELL_S[k] if pw) for k in range(1, 8)]
            sp, cp = mp.sin(psi), mp.cos(psi)

        def derivs(t):
            M = om * t + al
            if not elliptical:
                X, XM = mp.sin(M), mp.cos(M)
                return [k2 * (t + tau * X), k2 * f0 * X, k2 * f0 * tau * t * XM, k2 * f0 * tau * XM]
            co = [mp.cos(k * M) for k in range(8)]
            si = [mp.sin(k * M) for k in range(8)]
            cc = sum(C[k] * co[k] for k in range(8))
            ss = sum(S[k] * si[k] for k in range(1, 8))
            X, XM = sp * cc + cp * ss, sp * sum(-k * C[k] * si[k] for k in range(8)) + cp * sum(k * S[k] * co[k] for k in range(1, 8))
            Xp = cp * cc - sp * ss
            Xe = sp * sum(dC[k] * co[k] for k in range(8)) + cp * sum(dS[k] * si[k] for k in range(1, 8))
            return [k2 * (t + tau * X), k2 * f0 * X, k2 * f0 * tau * t * XM, k2 * f0 * tau * XM, k2 * f0 * tau * Xp, k2 * f0 * tau * Xe]

        nodes = mp.calculus.quadrature.GaussLegendre(mp.mp).calc_nodes(6, mp.mp.prec)      # 96 nodes on (-1, 1)
        panels = max(1, -(-int(n_quad) // 96))
        n = 6 if elliptical else 4
        mean = [mp.mpf(0)] * n
        mom = [[mp.mpf(0)] * n for _ in range(n)]
        for p in range(panels):
            a, b = t_obs * p / panels, t_obs * (p + 1) / panels
            for x, w in nodes:
                d = derivs((a + b) / 2 + (b - a) / 2 * x)
                ww = w / (2 * panels)
                for i in range(n):
                    mean[i] += ww * d[i]
                    for j in range(i, n):
                        mom[i][j] += ww * d[i] * d[j]
        g = mp.matrix(n, n)
        for i in range(n):
            for j in range(n):
                g[i, j] = mom[min(i, j)][max(i, j)] - mean[i] * mean[j]                      # eq 13
        gam = mp.matrix(n - 1, n - 1)
        for i in range(n - 1):
            for j in range(n - 1):
                gam[i, j] = g[i + 1, j + 1] - g[0, i + 1] * g[0, j + 1] / g[0, 0]              # eq 22
        return float(mp.sqrt(abs(mp.det(gam))))


def mismatch_direct(t_obs, phase_a, phase_b, n_quad=N_QUAD):
    """eq 12 (L92) from its definition: m = 1 - P(L, L') / P(L, L) with the detection statistic of a
    unit-amplitude monochromatic signal demodulated with the other phase model,
    P ~ |<exp(i (Phi_a - Phi_b))>_T|^2.  phase_a/b: callables t -> radians."""
    t, w = quadrature(t_obs, n_quad)
    d = (phase_a(t) - phase_b(t)).astype(LD)
    return float(1 - (np.sum(w * np.cos(d)) ** 2 + np.sum(w * np.sin(d)) ** 2))


# ----------------------------------------------------------------------------------------------
# eq 31, Table 1: the prior box
# ----------------------------------------------------------------------------------------------
def tau_max(omega, m_pulsar_min, m_comp_max, theta=1.0):
    """Upper limit of a sin(i)/c in lt-s for orbital angular velocity omega [rad/s]  (eq 31):
    theta G^(1/3) Omega^(-2/3) m_c / (c (m_p + m_c)^(2/3)), masses in solar masses (G M_sun / c^3 = T_SUN)."""
    return theta * T_SUN ** (1.0 / 3.0) * omega ** (-2.0 / 3.0) * m_comp_max / (m_pulsar_min + m_comp_max) ** (2.0 / 3.0)


def proposal(u, space):
    """Map uniforms u[0..5] in [0, 1) to a point of the prior box (Table 1):
    P_orb = P1 + u0 (P2 - P1), tau = u1 tau_max(Omega), alpha = 2 pi u2, psi = 2 pi u3, e = u4 e_max.
    Returns lam = (tau, Omega, alpha[, psi, e]) as float64 (the precision of the interface)."""
    p_orb = space["p_orb_min"] + float(u[0]) * (space["p_orb_max"] - space["p_orb_min"])
    omega = 2.0 * math.pi / p_orb
    tau = float(u[1]) * tau_max(omega, space["m_pulsar_min"], space["m_comp_max"], space.get("theta", 1.0))
    lam = [tau, omega, 2.0 * math.pi * float(u[2])]
    if space["elliptical"]:
        lam += [2.0 * math.pi * float(u[3]), float(u[4]) * space["e_max"]]
    return lam


def proposal_pdf(lam, space):
    """Density of `proposal` in the coordinates (tau, Omega, alpha[, psi, e]): P_orb uniform means
    q(Omega) = (P^2 / 2 pi) / (P2 - P1)."""
    omega = lam[1]
    p = 2.0 * math.pi / omega
    q = (p * p / (2.0 * math.pi)) / (space["p_orb_max"] - space["p_orb_min"])
    q /= tau_max(omega, space["m_pulsar_min"], space["m_comp_max"], space.get("theta", 1.0))
    q /= 2.0 * math.pi
    if space["elliptical"]:
        q /= 2.0 * math.pi * space["e_max"]
    return q


def template_of(lam, elliptical):
    """(P_orb, tau, phi0, e, omega) of include/tb.h from lam (alpha = phi0, psi = omega, L45)."""
    return (2.0 * math.pi / lam[1], lam[0], lam[2], lam[4] if elliptical else 0.0, lam[3] if elliptical else 0.0)


# ----------------------------------------------------------------------------------------------
# section 2.3 / 2.7: placement, volume, number of templates
# ----------------------------------------------------------------------------------------------
def generate(uniforms, space, rho_max, n_quad=N_QUAD, digits=None):
    """Rejection placement (G28): proposal i is accepted iff u_i5 * rho_max < rho(lam_i).
    uniforms: [n, 6].  Returns (accepted templates [k, 5], rho [n], accepted mask [n], volume estimate),
    the proper volume V = int rho d lam (eq 17) estimated as mean(rho_i / q(lam_i))."""
    ell = bool(space["elliptical"])
    rho = np.zeros(len(uniforms))
    vol = 0.0
    out, mask = [], np.zeros(len(uniforms), bool)
    for i, u in enumerate(uniforms):
        lam = proposal(u, space)
        rho[i] = density(space["f_max"], lam, space["t_obs"], ell, n_quad, digits)
        vol += rho[i] / proposal_pdf(lam, space)
        if float(u[5]) * rho_max < rho[i]:
            mask[i] = True
            out.append(template_of(lam, ell))
    return np.array(out, dtype=np.float64).reshape(-1, 5), rho, mask, vol / max(len(uniforms), 1)


def ball_volume(n):
    """C_n = pi^(n/2) / Gamma(n/2 + 1)  (eq 18)."""
    return math.pi ** (n / 2.0) / math.gamma(n / 2.0 + 1.0)


def n_templates(eta, m_star, n, volume, exact=True):
    """N_R(eta, m*, S_n): eq 20 (L131) or its large-volume expansion eq 21 (L136)."""
    x = m_star ** (n / 2.0) * ball_volume(n) / volume
    if exact:
        return math.log(1.0 - eta) / math.log1p(-x)
    return math.log(1.0 / (1.0 - eta)) / x
