"""ORACLE side of the steady-state shape measures and effective exponents (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Plain Python loops in fp64 written from the paper's definitions; shares nothing with
paper_1605_02620_b200/analysis.py.  P:n = /root/reference/PAPER.md line n.

  Eq. (13) P:180-184   Phi^n[phi] = <(phi - <phi>)^n>  over the distribution of the observable phi
  Eq. (14) P:186       S = <Phi^3> / <Phi^2>^(3/2)
  Eq. (15) P:188-190   Q = <Phi^4> / <Phi^2>^2 - 3
  Eq. (8)  P:92        alpha_eff = [ln W(L) - ln W(L/2)] / [ln L - ln(L/2)]
  Eq. (9)  P:94        beta_eff  = [ln W(t_i) - ln W(t_j)] / [ln t_i - ln t_j],  t_j = measured time nearest t_i / 2
  Eq. (10) P:97-101    t_{i+1} = (t_i + 10) e^m, m = 0.01, t_0 = 0  (rounded to the nearest integer, reading Q11)
  P:101 (reading Q9)   standard error of the mean sqrt((<x^2> - <x>^2) / (n - 1))

Pins (tests/test_analysis.py): a hand-worked sample, scipy.stats skew / kurtosis, closed forms of the exponential
distribution, exact power laws, the first Eq. (10) times computed by hand.
"""
import math


def central_moments(xs):
    """(mean, Phi^2, Phi^3, Phi^4) of a list of numbers: Eq. (13) with the empirical distribution."""
    n = len(xs)
    mean = 0.0
    for x in xs:
        mean += float(x)
    mean /= n
    p2 = p3 = p4 = 0.0
    for x in xs:
        d = float(x) - mean
        p2 += d * d
        p3 += d * d * d
        p4 += d * d * d * d
    return mean, p2 / n, p3 / n, p4 / n


def skewness_kurtosis(xs):
    """Eq. (14), (15) for one distribution sampled by xs (e.g. W^2 over realizations and times)."""
    _, p2, p3, p4 = central_moments(xs)
    return p3 / p2 ** 1.5, p4 / (p2 * p2) - 3.0


def height_skewness_kurtosis(per_surface):
    """Eq. (14), (15) with phi = h: per_surface = list of (Phi^2, Phi^3, Phi^4) of single surfaces (Eq. 13 over the
    sites of one surface); <.> averages over the surfaces."""
    n = len(per_surface)
    m2 = m3 = m4 = 0.0
    for (a, b, c) in per_surface:
        m2 += a
        m3 += b
        m4 += c
    m2, m3, m4 = m2 / n, m3 / n, m4 / n
    return m3 / m2 ** 1.5, m4 / (m2 * m2) - 3.0


def standard_error(xs):
    n = len(xs)
    s = s2 = 0.0
    for x in xs:
        s += float(x)
        s2 += float(x) * float(x)
    return math.sqrt(max(s2 / n - (s / n) ** 2, 0.0) / (n - 1))


def beta_eff(times, w2_mean):
    out = []
    for i in range(len(times)):
        if times[i] <= 1 or i == 0:
            continue
        best = None
        for j in range(i):
            if best is None or abs(times[j] - times[i] / 2.0) < abs(times[best] - times[i] / 2.0):
                best = j
        if times[best] <= 0 or times[best] >= times[i]:
            continue
        lw_i, lw_j = 0.5 * math.log(w2_mean[i]), 0.5 * math.log(w2_mean[best])
        out.append((times[i], (lw_i - lw_j) / (math.log(times[i]) - math.log(times[best]))))
    return out


def alpha_eff(sizes, w2_sat):
    out = []
    for i in range(1, len(sizes)):
        lw1, lw0 = 0.5 * math.log(w2_sat[i]), 0.5 * math.log(w2_sat[i - 1])
        out.append((sizes[i], (lw1 - lw0) / (math.log(sizes[i]) - math.log(sizes[i - 1]))))
    return out


def eq10_times(t_max, m=0.01):
    out, t = [], 0.0
    while True:
        t = (t + 10.0) * math.exp(m)
        ti = int(math.floor(t + 0.5))
        if ti > t_max:
            return out
        if not out or ti > out[-1]:
            out.append(ti)
