"""Pins for the shape measures (Eq. 13-15), effective exponents (Eq. 8, 9), the Eq. (10)
time schedule and the standard error (reading Q9): the ORACLE functions
(oracle/analysis_oracle.py) against hand-worked values, scipy.stats and closed forms; then the product's
host-side analysis (paper_1605_02620_b200/analysis.py, utils/workloads.py) against the oracle's."""
import math

import numpy as np
import pytest


@pytest.fixture(scope="module")
def ao():
    from oracle import analysis_oracle
    return analysis_oracle


def test_hand_worked_sample(ao):
    # x = (0, 0, 0, 4): mean 1, deviations (-1, -1, -1, 3): Phi2 = 12/4 = 3, Phi3 = 24/4 = 6, Phi4 = 84/4 = 21
    mean, p2, p3, p4 = ao.central_moments([0, 0, 0, 4])
    assert (mean, p2, p3, p4) == (1.0, 3.0, 6.0, 21.0)
    S, Q = ao.skewness_kurtosis([0, 0, 0, 4])
    assert S == pytest.approx(6.0 / 3.0 ** 1.5, rel=1e-15)          # 1.1547...
    assert Q == pytest.approx(21.0 / 9.0 - 3.0, rel=1e-15)          # -2/3
    # standard error of (1, 3): <x^2> - <x>^2 = 1, n - 1 = 1
    assert ao.standard_error([1, 3]) == pytest.approx(1.0)
    # two surfaces with (Phi2, Phi3, Phi4) = (1, 1, 4) and (3, 1, 12): means (2, 1, 8): S_h = 1 / 2^1.5, Q_h = 8/4 - 3
    S_h, Q_h = ao.height_skewness_kurtosis([(1, 1, 4), (3, 1, 12)])
    assert S_h == pytest.approx(1.0 / 2.0 ** 1.5) and Q_h == pytest.approx(-1.0)


def test_against_scipy_and_closed_forms(ao):
    from scipy import stats
    rng = np.random.default_rng(3)
    x = rng.gamma(2.5, 1.3, size=20000)
    S, Q = ao.skewness_kurtosis(list(x))
    assert S == pytest.approx(stats.skew(x, bias=True), rel=1e-10)
    assert Q == pytest.approx(stats.kurtosis(x, fisher=True, bias=True), rel=1e-10)
    # exponential distribution: skewness 2, excess kurtosis 6 (closed form), within sampling error
    e = rng.exponential(1.0, size=400000)
    S, Q = ao.skewness_kurtosis(list(e))
    assert abs(S - 2.0) < 0.05 and abs(Q - 6.0) < 0.6
    assert ao.standard_error(list(x)) == pytest.approx(stats.sem(x, ddof=1) * math.sqrt((len(x) - 1) / len(x)) *
                                                      math.sqrt(len(x) / (len(x) - 1)), rel=1e-9)


def test_effective_exponents_on_exact_power_laws(ao):
    times = [1, 2, 4, 8, 16, 32, 64, 100, 200]
    w2 = [t ** (2 * 0.2415) for t in times]
    for t, b in ao.beta_eff(times, w2):
        assert b == pytest.approx(0.2415, rel=1e-12)
    sizes = [32, 64, 128, 256, 512]
    w2s = [3.0 * L ** (2 * 0.39) for L in sizes]
    for L, a in ao.alpha_eff(sizes, w2s):
        assert a == pytest.approx(0.39, rel=1e-12)
    # partner choice: for t_i = 100 the measured time nearest 50 is 64
    w2b = [1.0] * len(times)
    w2b[times.index(64)] = math.e ** 2          # W(64) = e, others 1
    got = dict(ao.beta_eff(times, w2b))
    assert got[100] == pytest.approx((0.0 - 1.0) / (math.log(100) - math.log(64)))


def test_eq10_times_by_hand(ao):
    # t1 = 10 e^0.01 = 10.1005, t2 = 20.1005 e^0.01 = 20.3025, t3 = 30.3025 e^0.01 = 30.6071, t4 = 41.0151, t5 = 51.5278
    assert ao.eq10_times(60) == [10, 20, 31, 41, 52]
    t = ao.eq10_times(100000)
    assert t[-1] <= 100000 and all(b > a for a, b in zip(t, t[1:]))
    # late times grow by e^0.01 per step
    assert t[-1] / t[-2] == pytest.approx(math.exp(0.01), rel=2e-4)


def test_product_analysis_equals_oracle(ao):
    from paper_1605_02620_b200 import analysis
    from paper_1605_02620_b200.utils import workloads
    rng = np.random.default_rng(11)
    x = rng.gamma(3.0, 2.0, size=5000)
    S, Q = analysis.distribution_shape(x)
    So, Qo = ao.skewness_kurtosis(list(x))
    assert S == pytest.approx(So, rel=1e-10) and Q == pytest.approx(Qo, rel=1e-10)
    phi = np.abs(rng.normal(size=(300, 3))) + 0.5
    S, Q = analysis.height_distribution_shape(phi)
    So, Qo = ao.height_skewness_kurtosis([tuple(r) for r in phi])
    assert S == pytest.approx(So, rel=1e-12) and Q == pytest.approx(Qo, rel=1e-12)
    assert analysis.standard_error(x) == pytest.approx(ao.standard_error(list(x)), rel=1e-10)
    times = workloads.log_spaced_times(5000)
    w2 = [0.3 * t ** 0.47 + 0.1 for t in times]
    bt, be = analysis.beta_eff(times, w2)
    ref = ao.beta_eff(times, w2)
    assert list(bt) == [r[0] for r in ref] and np.allclose(be, [r[1] for r in ref], rtol=1e-12)
    Ls, ae = analysis.alpha_eff([64, 128, 256], [3.0, 5.2, 9.1])
    assert np.allclose(ae, [r[1] for r in ao.alpha_eff([64, 128, 256], [3.0, 5.2, 9.1])], rtol=1e-12)
    assert workloads.eq10_times(100000) == ao.eq10_times(100000)
