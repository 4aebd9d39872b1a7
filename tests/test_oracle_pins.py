"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

PAPER.md prints no worked numerical example, so the pins are closed forms,
invariants, textbook special cases and brute force.
Each test names the passage it rests on.  None of them retypes the oracle's loop.
"""
import numpy as np
import pytest

import smre_inputs as si

C = lambda sides: si.thresholds(sides).astype(np.float64)


def all_window_ratio(oracle, x, sides, c):
    """max over every window (all shifts) of t_s / c_S (t_s: PAPER.md:93)."""
    return max(float(oracle.window_sums(x, int(s)).max()) / float(cs) for s, cs in zip(sides, c))


# ---- golden constants: threshold table of BASELINE.json, c_S = |S| + 2 sqrt(2|S|) -------------
def test_threshold_table_golden():
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "thresholds_sigma1.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    sides = np.array([int(r[0]) for r in rows])
    want = np.array([float(r[1]) for r in rows])
    np.testing.assert_allclose(si.thresholds(sides), want, rtol=2e-7)


# ---- P1: single ball, closed form (Eq. 14) ----------------------------------------
@pytest.mark.parametrize("s", [1, 2, 3, 5, 8])
def test_single_ball_closed_form(oracle, s):
    rng = np.random.default_rng(10 + s)
    y = 3.0 * rng.standard_normal((s, s))
    c = float(C([s])[0])
    x = oracle.project_std(y, [s], [c], 1) if s == 1 else oracle.dykstra_families(y, [(s, 0, 0, c)], 1)
    n2 = float((y * y).sum())
    want = y * min(1.0, np.sqrt(c / n2))
    np.testing.assert_allclose(x, want, rtol=1e-15, atol=0)
    if n2 > c:
        assert abs((x * x).sum() - c) < 1e-12 * c


# ---- P2: identity on feasible input, bit for bit (Eq. 14 else-branch; strict compare A5) -------
@pytest.mark.parametrize("variant", ["standard", "incomplete"])
def test_identity_on_feasible_input(oracle, variant):
    rng = np.random.default_rng(2)
    sides = np.arange(1, 9)
    y = 0.2 * rng.standard_normal((40, 37))          # every window far inside its ball
    assert all_window_ratio(oracle, y, sides, C(sides)) < 1.0
    x = oracle.project(y, sides, C(sides), 7, variant)
    assert np.array_equal(x, y)
    if variant == "standard":
        _, q = oracle.project_std(y, sides, C(sides), 3, return_q=True)
        assert not q.any()


def test_boundary_is_not_scaled(oracle):
    # ||y||^2 == c exactly -> "else" branch (strict >, PAPER.md:170 / 506)
    y = np.array([[3.0, 4.0]]).reshape(1, 2)
    x = oracle.dykstra_families(np.array([[3.0, 0.0], [0.0, 4.0]]), [(2, 0, 0, 25.0)], 3)
    assert np.array_equal(x, np.array([[3.0, 0.0], [0.0, 4.0]]))
    x0 = oracle.dykstra_families(np.zeros((4, 4)), [(2, 0, 0, 1.0), (1, 0, 0, 0.5)], 3)
    assert np.array_equal(x0, np.zeros((4, 4)))      # n2 = 0 never divides


# ---- P3: one family => one projection; later sweeps change nothing (Alg. 2) --------------------
@pytest.mark.parametrize("s,oy,ox", [(3, 1, 2), (4, 0, 3), (8, 5, 5)])
def test_one_family_is_one_projection(oracle, s, oy, ox):
    rng = np.random.default_rng(3)
    y = 2.5 * rng.standard_normal((29, 31))
    c = float(C([s])[0])
    x1 = oracle.dykstra_families(y, [(s, oy, ox, c)], 1)
    x9 = oracle.dykstra_families(y, [(s, oy, ox, c)], 9)
    np.testing.assert_allclose(x9, x1, rtol=0, atol=2e-15)
    want = y.copy()
    for wy in range(oy, 29 - s + 1, s):
        for wx in range(ox, 31 - s + 1, s):
            blk = y[wy:wy + s, wx:wx + s]
            want[wy:wy + s, wx:wx + s] = blk * min(1.0, np.sqrt(c / (blk * blk).sum()))
    np.testing.assert_allclose(x1, want, rtol=1e-15)
    # pixels outside every full window are untouched (reading A6)
    assert np.array_equal(x1[:oy], y[:oy]) and np.array_equal(x1[:, :ox], y[:, :ox])


# ---- P4: side 1 only == clip at +-sqrt(c_1) (Eq. 14 with |s| = 1) -------------------------------
@pytest.mark.parametrize("variant", ["standard", "incomplete"])
def test_side_one_is_clip(oracle, variant):
    rng = np.random.default_rng(4)
    y = 3.0 * rng.standard_normal((17, 23))
    c1 = float(C([1])[0])
    x = oracle.project(y, [1], [c1], 5, variant)
    np.testing.assert_allclose(x, np.clip(y, -np.sqrt(c1), np.sqrt(c1)), rtol=1e-15)
    assert abs(np.sqrt(c1) - 1.956637) < 1e-6


# ---- P5: conservation x + sum_f q_f == y after any number of sweeps (Listing 3: 477/502/510) ---
def test_conservation_invariant(oracle):
    w = si.config(0)
    for n in (1, 2, 13):
        x, q = oracle.project_std(w.y, w.sides, w.c, n, return_q=True)
        assert np.abs(x + q.sum(axis=0) - w.y.astype(np.float64)).max() < 1e-13
    assert q.shape[0] == 30


# ---- P6: feasibility in the limit ------------------------------------------------
def test_feasible_in_the_limit_tiny(oracle):
    rng = np.random.default_rng(6)
    y = 2.0 * rng.standard_normal((7, 8))
    sides = [1, 2, 3]
    x = oracle.project_std(y, sides, C(sides), 20000)
    assert all_window_ratio(oracle, x, sides, C(sides)) <= 1.0 + 1e-9


def test_violation_decreases_with_sweeps_c0(oracle):
    w = si.config(0)
    r = [all_window_ratio(oracle, oracle.project_std(w.y, w.sides, w.c, n), w.sides, w.c.astype(float))
         for n in (50, 200, 1000)]
    assert r[0] > r[1] > r[2] > 1.0 - 1e-12
    assert r[0] < 1.05 and r[1] < 1.0 + 1e-5 and r[2] < 1.0 + 1e-12


# ---- helpers for the optimality pins --------------------------------------------------------------
def feasible_scale(oracle, w, sides, c):
    """tau_G is star-shaped about 0: scale any w into it."""
    r = all_window_ratio(oracle, w, sides, c)
    return w * min(1.0, 1.0 / np.sqrt(r)) if r > 0 else w


# ---- P7: variational inequality <y - x*, z - x*> <= 0 for feasible z (Eq. 13) ----
def test_variational_inequality_at_convergence(oracle):
    rng = np.random.default_rng(7)
    sides = [1, 2, 3]
    c = C(sides)
    y = 2.5 * rng.standard_normal((6, 6))
    x = oracle.project_std(y, sides, c, 50000)
    worst = -np.inf
    for k in range(400):
        z = rng.standard_normal((6, 6)) * rng.uniform(0.1, 4.0)
        if k % 4 == 0:
            z = x + 0.3 * rng.standard_normal((6, 6))      # near the solution
        if k % 4 == 1:
            z = y + 0.3 * rng.standard_normal((6, 6))      # towards y
        z = feasible_scale(oracle, z, sides, c)
        worst = max(worst, float(((y - x) * (z - x)).sum()))
    assert worst <= 1e-7
    # and x* is not just any feasible point: it is closer to y than every sampled feasible z
    assert all_window_ratio(oracle, x, sides, c) <= 1 + 1e-9


# ---- P8: KKT structure: y - x* = sum_f q_f, q_{f,S} = lambda x*_S, lambda >= 0, 0 if inactive ---
def test_kkt_structure_at_convergence(oracle):
    rng = np.random.default_rng(8)
    sides = [1, 2, 3]
    c = C(sides)
    y = 2.5 * rng.standard_normal((6, 7))
    fams = oracle.std_family_list(sides, c)
    x, q = oracle.dykstra_families(y, fams, 50000, return_q=True)
    np.testing.assert_allclose(x + q.sum(0), y, atol=1e-12)
    n_active = 0
    for f, (s, oy, ox, cs) in enumerate(fams):
        for wy in range(oy, 6 - s + 1, s):
            for wx in range(ox, 7 - s + 1, s):
                xb = x[wy:wy + s, wx:wx + s].ravel()
                qb = q[f, wy:wy + s, wx:wx + s].ravel()
                if not qb.any():
                    continue
                n_active += 1
                lam = qb @ xb / (xb @ xb)
                assert lam > 0
                np.testing.assert_allclose(qb, lam * xb, atol=1e-9)       # parallel to x*_S
                assert abs(xb @ xb - cs) < 1e-6 * cs                      # multiplier only on tight balls
    assert n_active > 0


# ---- P9: brute force with an independent generic solver (Eq. 13) ---------------------------------
@pytest.mark.parametrize("H,W,sides,seed", [(4, 4, [1, 2], 0), (5, 5, [1, 2, 3], 1), (6, 5, [2, 3], 2)])
def test_brute_force_slsqp(oracle, H, W, sides, seed):
    from scipy.optimize import minimize
    rng = np.random.default_rng(90 + seed)
    y = 2.5 * rng.standard_normal((H, W))
    c = C(sides)
    wins = [(s, wy, wx, cs) for s, cs in zip(sides, c)
            for wy in range(H - s + 1) for wx in range(W - s + 1)]

    def cons(v):
        X = v.reshape(H, W)
        return np.array([cs - (X[wy:wy + s, wx:wx + s] ** 2).sum() for s, wy, wx, cs in wins])

    def cons_jac(v):
        X = v.reshape(H, W)
        J = np.zeros((len(wins), H * W))
        for k, (s, wy, wx, _) in enumerate(wins):
            G = np.zeros((H, W))
            G[wy:wy + s, wx:wx + s] = -2.0 * X[wy:wy + s, wx:wx + s]
            J[k] = G.ravel()
        return J

    res = minimize(lambda v: 0.5 * ((v - y.ravel()) ** 2).sum(), np.zeros(H * W),
                   jac=lambda v: v - y.ravel(), method="SLSQP",
                   constraints=[{"type": "ineq", "fun": cons, "jac": cons_jac}],
                   options={"ftol": 1e-15, "maxiter": 2000})
    # status 8 = line search cannot improve any further at ftol = 1e-15: already at the optimum
    assert res.status in (0, 8), res.message
    assert cons(res.x).min() > -1e-9
    x = oracle.project_std(y, sides, c, 100000)
    np.testing.assert_allclose(x, res.x.reshape(H, W), atol=1e-6)


# ---- P10: box cap ball, textbook closed form (KKT of Eq. 13) -------------------------------------
@pytest.mark.parametrize("s", [3, 4, 6])
def test_box_and_ball_closed_form(oracle, s):
    rng = np.random.default_rng(100 + s)
    y = 4.0 * rng.standard_normal((s, s))
    c1 = float(C([1])[0])
    b = np.sqrt(c1)
    cs = 0.8 * float((np.clip(y, -b, b) ** 2).sum())  # ball tight enough that both constraints bind
    g = lambda lam: (np.clip(y / (1 + lam), -b, b) ** 2).sum() - cs
    assert g(0.0) > 0
    lo, hi = 0.0, 1.0
    while g(hi) > 0:
        hi *= 2
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if g(mid) > 0 else (lo, mid)
    want = np.clip(y / (1 + hi), -b, b)
    x = oracle.project_std(y, [1, s], [c1, cs], 20000)
    np.testing.assert_allclose(x, want, atol=1e-10)
    assert (np.abs(want) == b).any() and (np.abs(want) < b).any()


# ---- P11: symmetries that hold at any sweep count (Eq. 5, 14) ------------------------------------
@pytest.mark.parametrize("variant", ["standard", "incomplete"])
def test_odd_and_homogeneous(oracle, variant):
    w = si.config(0)
    y = w.y.astype(np.float64)[:32, :40]
    sides, c = w.sides, w.c.astype(np.float64)
    x = oracle.project(y, sides, c, 5, variant)
    assert np.array_equal(oracle.project(-y, sides, c, 5, variant), -x)
    assert np.array_equal(oracle.project(4.0 * y, sides, 16.0 * c, 5, variant), 4.0 * x)


def test_transpose_equivariance_at_convergence(oracle):
    rng = np.random.default_rng(11)
    y = 2.5 * rng.standard_normal((6, 7))
    sides = [1, 2, 3]
    a = oracle.project_std(y, sides, C(sides), 50000)
    b = oracle.project_std(y.T.copy(), sides, C(sides), 50000).T
    np.testing.assert_allclose(a, b, atol=1e-9)
    f = oracle.project_std(y[::-1, ::-1].copy(), sides, C(sides), 50000)[::-1, ::-1]
    np.testing.assert_allclose(a, f, atol=1e-9)


# ---- the checker itself: t_s of every window at every shift ----------------------------
# smre_oracle_window_sums forms the violated-window sets of the parity protocol and every feasibility pin
# above, so it gets its own pin: an independent strided-view sum (numpy sliding_window_view, no loop of the
# oracle retyped), the exact output shape (H-s+1, W-s+1) and the LAST row / column of windows on a ragged
# image, whose values are chosen so that a dropped or shifted origin cannot go unnoticed.
@pytest.mark.parametrize("H,W", [(23, 31), (8, 8), (9, 17)])
def test_window_sums_checker_against_sliding_view(oracle, H, W):
    from numpy.lib.stride_tricks import sliding_window_view
    rng = np.random.default_rng(H * 100 + W)
    x = rng.standard_normal((H, W))
    x[-1, :] += 7.0          # the last row and column dominate every window that contains them
    x[:, -1] -= 5.0
    for s in range(1, min(H, W, 8) + 1):
        got = oracle.window_sums(x, s)
        assert got.shape == (H - s + 1, W - s + 1)
        want = (sliding_window_view(x, (s, s)) ** 2).sum(axis=(2, 3))
        np.testing.assert_allclose(got, want, rtol=1e-13, atol=0)
        # origin (wy, wx) means rows wy..wy+s-1, columns wx..wx+s-1: a one-hot image has exactly s*s windows
        # containing the pixel, at origins (r-s+1..r, c-s+1..c) clipped to the image
        e = np.zeros((H, W))
        r, c0 = H - 1, W - 2
        e[r, c0] = 3.0
        t = oracle.window_sums(e, s)
        hit = np.argwhere(t > 0)
        assert (t[t > 0] == 9.0).all()
        assert hit[:, 0].min() == max(0, r - s + 1) and hit[:, 0].max() == min(r, H - s)
        assert hit[:, 1].min() == max(0, c0 - s + 1) and hit[:, 1].max() == min(c0, W - s)
