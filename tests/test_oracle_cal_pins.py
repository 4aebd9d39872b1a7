"""Pins of the oracle's threshold calibration (CPU only; sec. 2.1, lines 89-113).

Q_Omega = max_s ((t_s)^(1/4) - mu_s) / sigma_s over every window of every side; c_s(alpha) = 1 / (q_alpha sigma_s + mu_s)^4.
Pinned by closed forms (constant and one-hot images), an independent strided-view evaluation, the identity that ties
the thresholds back to Q (max_s c_s t_s = 1 where q_alpha = Q), the order-statistic definition of the quantile and
the statistics the transform is built on (fourth root of a chi-square is about N(mu_s, sigma_s^2)).
"""
import numpy as np
import pytest
from numpy.lib.stride_tricks import sliding_window_view


def mu(s):
    return (s * s - 0.5) ** 0.25


def sigma(s):
    return np.sqrt(1.0 / (8.0 * np.sqrt(s * s)))


def q_numpy(x, sides):
    return max((((sliding_window_view(x, (s, s)) ** 2).sum(axis=(2, 3)) ** 0.25 - mu(s)) / sigma(s)).max() for s in sides)


def test_constant_and_one_hot_images_closed_form(oracle):
    sides = [1, 2, 3, 5, 8]
    x = np.full((13, 17), 1.7)                                   # t_s = |s| v^2 for every window
    want = max(((s * s * 1.7 ** 2) ** 0.25 - mu(s)) / sigma(s) for s in sides)
    assert abs(oracle.q_stat(x, sides) - want) < 1e-12
    e = np.zeros((13, 17))
    e[12, 16] = 9.0                                              # the corner pixel: in exactly one window per side
    want = max((3.0 - mu(s)) / sigma(s) for s in sides)          # t = 81 -> fourth root 3; all other windows are < 0
    assert abs(oracle.q_stat(e, sides) - want) < 1e-12
    z = np.zeros((6, 6))                                         # all t = 0: Q = max_s (-mu_s / sigma_s)
    assert abs(oracle.q_stat(z, [2, 4]) - max(-mu(s) / sigma(s) for s in (2, 4))) < 1e-12


@pytest.mark.parametrize("H,W,sides", [(23, 31, [1, 2, 3, 4, 5, 6, 7, 8]), (16, 16, [16]), (20, 9, [3, 9]), (40, 37, [2, 11])])
def test_q_against_strided_view(oracle, H, W, sides):
    rng = np.random.default_rng(H + W)
    x = rng.standard_normal((H, W))
    x[-1, :] *= 3.0                                              # the last row / column matter
    x[:, -1] *= 2.5
    assert abs(oracle.q_stat(x, sides) - q_numpy(x, sides)) < 1e-11
    stack = rng.standard_normal((3, H, W))
    np.testing.assert_allclose(oracle.q_stat(stack, sides), [q_numpy(f, sides) for f in stack], rtol=0, atol=1e-11)


def test_thresholds_tie_back_to_q(oracle):
    """With q_alpha = Q(x) the worst window of x sits exactly on its constraint: max_s c_s t_s = 1,
    in this library's convention max_S t_S / c_S = 1; a larger quantile makes x feasible, a smaller one infeasible."""
    rng = np.random.default_rng(4)
    sides = [1, 2, 3, 4, 6]
    x = rng.standard_normal((19, 22))
    Q = oracle.q_stat(x, sides)
    for dq, cmp in ((0.0, "eq"), (0.05, "lt"), (-0.05, "gt")):
        qa, c = oracle.thresholds_from_q([Q + dq], 1.0, sides)
        assert qa == Q + dq
        worst = max(float(oracle.window_sums(x, s).max()) / float(cs) for s, cs in zip(sides, c))
        assert {"eq": abs(worst - 1.0) < 1e-12, "lt": worst < 1.0, "gt": worst > 1.0}[cmp]
    np.testing.assert_allclose(c, [((Q - 0.05) * sigma(s) + mu(s)) ** 4 for s in sides], rtol=1e-14)


def test_quantile_is_the_order_statistic(oracle):
    rng = np.random.default_rng(5)
    q = rng.standard_normal(37)
    srt = np.sort(q)
    for alpha in (0.01, 0.5, 0.9, 0.95, 1.0, 1 / 37, 2 / 37 + 1e-9):
        k = min(37, max(1, int(np.ceil(alpha * 37))))
        assert oracle.thresholds_from_q(q, alpha, [3])[0] == srt[k - 1]
    qs = [oracle.thresholds_from_q(q, a, [3])[0] for a in (0.1, 0.3, 0.6, 0.9)]
    assert qs == sorted(qs)
    # a larger quantile gives larger thresholds, side by side
    c1 = oracle.thresholds_from_q(q, 0.3, [1, 4, 9])[1]
    c2 = oracle.thresholds_from_q(q, 0.9, [1, 4, 9])[1]
    assert (c2 > c1).all()


def test_fourth_root_transform_statistics(oracle):
    """(t_s)^(1/4) of white noise is about N(mu_s, sigma_s^2): the standardised window statistic has
    mean ~ 0 and variance ~ 1 for every side -- wrong |s| (side instead of side^2) or a wrong constant fails."""
    rng = np.random.default_rng(6)
    x = rng.standard_normal((256, 256))
    for s in (2, 4, 8, 16):
        t = oracle.window_sums(x, s)[::s, ::s]                   # disjoint windows: independent samples
        z = (t ** 0.25 - mu(s)) / sigma(s)
        assert abs(z.mean()) < 0.12 and abs(z.var() - 1.0) < 0.2, (s, z.mean(), z.var())
    # and the quantile of Q on pure noise is a usable threshold level: about a fraction alpha of fresh noise images
    # are feasible for the thresholds it gives
    sides = [1, 2, 4]
    Q = oracle.q_stat(rng.standard_normal((200, 24, 24)), sides)
    qa, c = oracle.thresholds_from_q(Q, 0.8, sides)
    fresh = oracle.q_stat(rng.standard_normal((200, 24, 24)), sides)
    assert 0.65 < (fresh <= qa).mean() < 0.92


# ---- second-order SOFI cumulant (Eq. 19) --------------------------------------------------
def test_cumulant2_closed_forms(oracle):
    rng = np.random.default_rng(12)
    # a constant pixel has no fluctuation; a pixel that blinks between a and b half of the time has ((a - b) / 2)^2
    n, H, W = 8, 3, 4
    s = np.full((n, H, W), 2.5)
    s[::2, 1, 2] = 7.0
    s[1::2, 1, 2] = 1.0
    c2 = oracle.cumulant2(s)
    want = np.zeros((H, W))
    want[1, 2] = 9.0
    np.testing.assert_allclose(c2, want, atol=1e-13)
    # the population variance of numpy, shift invariance (cumulants of order >= 2 ignore a constant background) and
    # the quadratic scaling with the brightness
    s = rng.standard_normal((50, 6, 5)) * rng.uniform(0.5, 2.0, (1, 6, 5)) + 3.0
    c2 = oracle.cumulant2(s)
    np.testing.assert_allclose(c2, s.var(axis=0), rtol=1e-12)
    np.testing.assert_allclose(oracle.cumulant2(s + 100.0), c2, rtol=1e-9)
    np.testing.assert_allclose(oracle.cumulant2(3.0 * s), 9.0 * c2, rtol=1e-12)
    assert (c2 >= 0).all()
