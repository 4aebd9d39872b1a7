"""Pins of the oracle's ADMM around the projection (CPU only; Alg. 1,
Eq. 9-13; readings A-ADMM-1..9 of DESIGN.md).

What the paper fixes is the problem (Eq. 10) and the form of the updates; the pins therefore check the oracle against
the PROBLEM, not against a retyped loop: the limit for an identity PSF is the Euclidean projection (pinned oracle
function), the limit with inactive constraints is x = 0, the limit with a blur satisfies the KKT system of Eq. 10 and
agrees with a general-purpose constrained solver on a tiny image.  The PSF operator is pinned against scipy's
gaussian_filter and the plain 2-D definition.
"""
import numpy as np
import pytest

import smre_inputs as si

PAPER = dict(rho1=6.192, rho2=1.8, alpha1=1.2, alpha2=0.12, lam=1.0)       # App. B


def run(oracle, I, sides, c, sigma, gamma=8.0, delta=1e-10, max_iter=4000, variant=0, n_sweeps=200, **kw):
    p = dict(PAPER)
    p.update(kw)
    return oracle.admm(I, sides, c, variant, n_sweeps, sigma, p["rho1"], p["rho2"], p["alpha1"], p["alpha2"], p["lam"],
                       gamma, delta, max_iter)


# ---- the PSF operator -------------------------------------------------------------------------------------
@pytest.mark.parametrize("sigma", [0.6, 1.0, 1.5, 2.2])
def test_gauss_conv_against_scipy(oracle, sigma):
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(1)
    x = rng.standard_normal((19, 26))
    radius = int(np.ceil(3 * sigma))
    want = ndi.gaussian_filter(x, sigma, mode="constant", cval=0.0, truncate=(radius + 0.25) / sigma)
    np.testing.assert_allclose(oracle.gauss_conv(x, sigma), want, rtol=0, atol=1e-13)
    taps = oracle.gauss_taps(sigma)
    assert len(taps) == 2 * radius + 1 and abs(taps.sum() - 1.0) < 1e-15 and np.allclose(taps, taps[::-1])


def test_gauss_conv_definition_adjoint_and_special_cases(oracle):
    rng = np.random.default_rng(2)
    H, W, sigma = 7, 9, 0.8
    x = rng.standard_normal((H, W))
    t = oracle.gauss_taps(sigma)
    r = len(t) // 2
    want = np.zeros((H, W))                                       # the plain 2-D definition, zero outside
    for y in range(H):
        for c in range(W):
            for dy in range(-r, r + 1):
                for dx in range(-r, r + 1):
                    if 0 <= y + dy < H and 0 <= c + dx < W:
                        want[y, c] += t[dy + r] * t[dx + r] * x[y + dy, c + dx]
    np.testing.assert_allclose(oracle.gauss_conv(x, sigma), want, atol=1e-14)
    # A is symmetric (Eq. 11 uses A^T *): <A u, v> = <u, A v>, also next to the border
    u, v = rng.standard_normal((2, H, W))
    assert abs((oracle.gauss_conv(u, sigma) * v).sum() - (u * oracle.gauss_conv(v, sigma)).sum()) < 1e-12
    # sigma = 0 is the identity; a one-hot image gives the outer product of the taps
    assert np.array_equal(oracle.gauss_conv(x, 0.0), x)
    e = np.zeros((H, W))
    e[3, 4] = 1.0
    np.testing.assert_allclose(oracle.gauss_conv(e, sigma)[3 - r:3 + r + 1, 4 - r:4 + r + 1], np.outer(t, t), atol=1e-16)
    # a constant image stays constant away from the border and loses mass at it
    out = oracle.gauss_conv(np.ones((12, 12)), sigma)
    assert np.allclose(out[r:-r, r:-r], 1.0) and abs(out[0, 0] - t[r:].sum() ** 2) < 1e-15 and out[0, 0] < 0.6


# ---- the limit is the solution of Eq. 10 -------------------------------------------------------------------
@pytest.mark.parametrize("gamma", [4.0, 8.0, 20.0])
def test_identity_psf_reaches_the_projection(oracle, gamma):
    """A = identity: Eq. 10 is  min_{eps in C} (lambda / 2) ||I - eps||^2, so eps* = P_C(I) (the Euclidean projection,
    a pinned oracle function) and x* = I - P_C(I), whatever gamma and the penalty parameters are."""
    rng = np.random.default_rng(0)
    I = rng.standard_normal((24, 28)) + 2.0
    sides = [1, 2, 4]
    c = si.thresholds(sides).astype(np.float64)
    P = oracle.project_std(I, sides, c, 3000)
    assert np.abs(I - P).max() > 1.0                              # the constraints bite
    r = run(oracle, I, sides, c, 0.0, gamma=gamma)
    assert 50 < r["iters"] < 4000
    np.testing.assert_allclose(r["eps"], P, atol=1e-6)
    np.testing.assert_allclose(r["x"], I - P, atol=1e-6)
    np.testing.assert_allclose(r["z"], r["x"], atol=1e-8)
    r2 = run(oracle, I, sides, c, 0.0, gamma=gamma, rho1=3.0, rho2=0.7, alpha1=0.9, alpha2=0.3)
    np.testing.assert_allclose(r2["x"], I - P, atol=1e-6)


def test_inactive_constraints_give_zero(oracle):
    """Thresholds so large that every residual is feasible: eps is free, the minimiser of (lambda/2)||x||^2 is x = 0
    and the residual takes the whole image."""
    rng = np.random.default_rng(3)
    I = rng.standard_normal((16, 18)) + 1.0
    r = run(oracle, I, [1, 2, 3], np.full(3, 1e12), 1.0, delta=1e-11)
    assert np.abs(r["x"]).max() < 1e-8 and np.abs(r["eps"] - I).max() < 1e-8


def test_kkt_system_with_blur(oracle):
    """With a PSF the limit satisfies the KKT system of Eq. 10: both constraints hold, lambda z = Y2 (stationarity in
    z), A^T Y1 = Y2 (stationarity in x) and eps = P_C(eps + Y1 / rho1) (Y1 lies in the normal cone of C at eps)."""
    rng = np.random.default_rng(4)
    I = oracle.gauss_conv(3.0 * (rng.random((20, 22)) > 0.7), 1.0) + 0.4 * rng.standard_normal((20, 22))
    sides = [1, 2, 3, 4]
    c = (0.4 ** 2) * si.thresholds(sides).astype(np.float64)
    for variant in (0, 1):
        sd = sides if variant == 0 else [1, 2, 4]
        cc = c if variant == 0 else (0.4 ** 2) * si.thresholds(sd).astype(np.float64)
        r = run(oracle, I, sd, cc, 1.0, gamma=8.0, delta=1e-9, max_iter=20000, variant=variant, n_sweeps=300)
        assert r["iters"] < 20000
        x, eps, z, Y1, Y2 = r["x"], r["eps"], r["z"], r["Y1"], r["Y2"]
        assert np.abs(I - oracle.gauss_conv(x, 1.0) - eps).max() < 1e-7
        assert np.abs(x - z).max() < 1e-7
        assert np.abs(PAPER["lam"] * z - Y2).max() < 1e-6
        assert np.abs(oracle.gauss_conv(Y1, 1.0) - Y2).max() < 1e-6
        if variant == 0:                                          # the standard variant's P_G is the projection
            again = oracle.project_std(eps + Y1 / PAPER["rho1"], sd, cc, 3000)
            assert np.abs(again - eps).max() < 1e-5
            worst = max(float(oracle.window_sums(eps, s).max()) / float(cs) for s, cs in zip(sd, cc))
            assert worst < 1.0 + 1e-4 and np.abs(x).max() > 0.1   # feasible residual (up to the 300 sweeps of the
                                                                  # inner projection), a non-trivial estimate


def test_tiny_problem_against_a_general_solver(oracle):
    """6 x 6, sides 1-2, sigma = 0.7: minimise (lambda/2)||x||^2 subject to every window of I - A x inside its ball
    with scipy's SLSQP (no ADMM, no Dykstra)."""
    opt = pytest.importorskip("scipy.optimize")
    rng = np.random.default_rng(5)
    H = W = 6
    sigma, sides = 0.7, [1, 2]
    I = 1.5 + rng.standard_normal((H, W))
    c = 0.3 * si.thresholds(sides).astype(np.float64)
    A = np.zeros((H * W, H * W))                                  # the operator as a matrix, column by column
    for k in range(H * W):
        e = np.zeros(H * W)
        e[k] = 1.0
        A[:, k] = oracle.gauss_conv(e.reshape(H, W), sigma).ravel()
    wins = [(s, cs, y, x) for s, cs in zip(sides, c) for y in range(H - s + 1) for x in range(W - s + 1)]

    def cons(xv):
        eps = (I.ravel() - A @ xv).reshape(H, W)
        return np.array([cs - (eps[y:y + s, x:x + s] ** 2).sum() for s, cs, y, x in wins])

    def cjac(xv):
        eps = (I.ravel() - A @ xv).reshape(H, W)
        J = np.zeros((len(wins), H * W))
        for k, (s, cs, y, x) in enumerate(wins):
            m = np.zeros((H, W))
            m[y:y + s, x:x + s] = eps[y:y + s, x:x + s]
            J[k] = 2 * (A.T @ m.ravel())
        return J

    best = None
    for x0 in (np.zeros(H * W), I.ravel().copy(), 0.5 * I.ravel()):      # three starts, one answer
        res = opt.minimize(lambda v: 0.5 * (v ** 2).sum(), x0, jac=lambda v: v, method="SLSQP",
                           constraints=[{"type": "ineq", "fun": cons, "jac": cjac}],
                           options={"maxiter": 2000, "ftol": 1e-15})
        # (SLSQP ends with status 8, "positive directional derivative", once it cannot improve any more)
        assert res.status in (0, 8) and cons(res.x).min() > -1e-8
        assert best is None or abs(res.fun - best.fun) < 1e-8
        best = res
    res = best
    r = run(oracle, I, sides, c, sigma, gamma=8.0, delta=1e-11, max_iter=50000, n_sweeps=2000)
    assert r["iters"] < 50000
    assert abs(0.5 * (r["x"] ** 2).sum() - res.fun) < 1e-5 * max(1.0, res.fun)
    np.testing.assert_allclose(r["x"].ravel(), res.x, atol=2e-4)


# ---- the loop itself: first iterate, stop rule ----------------------------------------------------------------
def test_first_iterate_and_stop_rule(oracle):
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(6)
    I = rng.standard_normal((15, 17)) + 2.0
    sides = [1, 2, 4]
    c = si.thresholds(sides).astype(np.float64)
    sigma, gamma = 1.0, 8.0
    A = lambda u: ndi.gaussian_filter(u, sigma, mode="constant", truncate=3.25)
    # from x_0 = z_0 = 0, eps_0 = 0, Y = 0:  x_1 = rho1 A^T I / (2 gamma), eps_1 = P_G(I - A x_1), z_1 = rho2 x_1 / (lambda + rho2)
    r1 = run(oracle, I, sides, c, sigma, gamma=gamma, max_iter=1)
    x1 = PAPER["rho1"] * A(I) / (2 * gamma)
    np.testing.assert_allclose(r1["x"], x1, atol=1e-13)
    np.testing.assert_allclose(r1["eps"], oracle.project_std(I - A(x1), sides, c, 200), atol=1e-12)
    np.testing.assert_allclose(r1["z"], PAPER["rho2"] * x1 / (PAPER["lam"] + PAPER["rho2"]), atol=1e-13)
    np.testing.assert_allclose(r1["Y1"], PAPER["alpha1"] * (I - A(x1) - r1["eps"]), atol=1e-12)
    np.testing.assert_allclose(r1["Y2"], PAPER["alpha2"] * (x1 - r1["z"]), atol=1e-13)
    assert r1["iters"] == 1 and abs(r1["hist"][0, 0] - np.linalg.norm(x1)) < 1e-12
    # the loop ends with the first iteration in which BOTH norms are <= delta, and never before
    delta = 1e-3                                                  # App. B: tolerance = 1e-3
    r = run(oracle, I, sides, c, sigma, gamma=gamma, delta=delta, max_iter=5000)
    h = r["hist"]
    assert 1 < r["iters"] < 5000 and len(h) == r["iters"]
    small = (h[:, 0] <= delta) & (h[:, 1] <= delta)
    assert small[-1] and not small[:-1].any()
    # a run capped below that count returns exactly that many iterations and the same iterates on the way
    k = r["iters"] // 2
    rk = run(oracle, I, sides, c, sigma, gamma=gamma, delta=delta, max_iter=k)
    assert rk["iters"] == k and np.array_equal(rk["hist"], h[:k])
    # the count does not increase with delta
    its = [run(oracle, I, sides, c, sigma, gamma=gamma, delta=d, max_iter=5000)["iters"] for d in (1e-6, 1e-4, 1e-2)]
    assert its[0] >= its[1] >= its[2] > 1
