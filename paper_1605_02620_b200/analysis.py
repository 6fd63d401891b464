"""Host-side analysis of what the C ABI returns (SURVEY layer L5; S 8(f) NEXT-2 and NEXT-3): shape measures of
the width and height distributions (Eq. 13-15), effective exponents (Eq. 8, 9), the 1-sigma standard error.

Everything on the hot path runs in the CUDA kernels; these functions only combine the R per-realization numbers
(W^2 from rsos_width, Phi^2..Phi^4 from rsos_height_moments) that the library hands back.  numpy, fp64.
Citations: P:n = PAPER.md line n; Q = readings of DESIGN.md section 3.  Imports nothing from oracle/.
"""
import numpy as np


def standard_error(x):
    """1-sigma standard error of the mean (reading Q9): sqrt((<x^2> - <x>^2) / (n - 1))."""
    x = np.asarray(x, dtype=np.float64).ravel()
    if x.size < 2:
        return float("nan")
    return float(np.sqrt(max(np.mean(x * x) - np.mean(x) ** 2, 0.0) / (x.size - 1)))


def distribution_shape(samples):
    """Skewness S and kurtosis Q (Eq. 14, 15) of the distribution P(phi) of a scalar interface observable
    phi sampled over realizations (and times), e.g. phi = W^2(L) in the steady state (S = 1.70(1), Q = 5.38(4)):
    Phi^n = <(phi - <phi>)^n> (Eq. 13), S = Phi^3 / (Phi^2)^(3/2), Q = Phi^4 / (Phi^2)^2 - 3."""
    x = np.asarray(samples, dtype=np.float64).ravel()
    d = x - x.mean()
    p2, p3, p4 = np.mean(d ** 2), np.mean(d ** 3), np.mean(d ** 4)
    return float(p3 / p2 ** 1.5), float(p4 / p2 ** 2 - 3.0)


def height_distribution_shape(phi):
    """S_h and Q_h (Eq. 14, 15 with phi = h; S_h = 0.270(5), Q_h = 0.15(1)) from the per-surface central
    moments Phi^2, Phi^3, Phi^4 of rsos_height_moments (array [..., 3]), <.> = average over surfaces and times:
    S_h = <Phi^3> / <Phi^2>^(3/2), Q_h = <Phi^4> / <Phi^2>^2 - 3."""
    phi = np.asarray(phi, dtype=np.float64).reshape(-1, 3)
    m2, m3, m4 = phi[:, 0].mean(), phi[:, 1].mean(), phi[:, 2].mean()
    return float(m3 / m2 ** 1.5), float(m4 / m2 ** 2 - 3.0)


def beta_eff(times, w2_mean):
    """Effective growth exponent, Eq. (9) (the argument labels are garbled in the source, reading Q10):
    beta_eff(t_i) = [ln W(t_i) - ln W(t_j)] / [ln t_i - ln t_j] with W = sqrt(<W^2>) and t_j the measurement time
    nearest to t_i / 2 (t_j < t_i).  Returns (t_i, beta_eff) for every i that has such a partner."""
    t = np.asarray(times, dtype=np.float64)
    w = 0.5 * np.log(np.asarray(w2_mean, dtype=np.float64))
    out_t, out_b = [], []
    for i in range(len(t)):
        if t[i] <= 1:
            continue
        j = int(np.argmin(np.abs(t[:i] - t[i] / 2.0))) if i else -1
        if j < 0 or t[j] <= 0 or t[j] >= t[i]:
            continue
        out_t.append(t[i])
        out_b.append((w[i] - w[j]) / (np.log(t[i]) - np.log(t[j])))
    return np.array(out_t), np.array(out_b)


def alpha_eff(sizes, w2_sat):
    """Effective roughness exponent, Eq. (8): alpha_eff = [ln W(L) - ln W(L/2)] / [ln L - ln(L/2)] for
    consecutive system sizes (sorted ascending), W = sqrt(<W^2>_sat).  Returns (L, alpha_eff(L)) for L = sizes[1:]."""
    L = np.asarray(sizes, dtype=np.float64)
    w = 0.5 * np.log(np.asarray(w2_sat, dtype=np.float64))
    return L[1:], (w[1:] - w[:-1]) / (np.log(L[1:]) - np.log(L[:-1]))
