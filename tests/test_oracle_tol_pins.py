"""Pins of the oracle's convergence-controlled modes (CPU only).

Standard variant: Alg. 2's stop rule ||x_r - x_{r-1}||^2 <= delta per sweep (reading A4').
Incomplete variant: Listing 3's per-tile rule sum |e_old - e_new| <= tol * L^2 (reading A-ICD-16).
The pins do not retype the oracle's loops: the stop sweep is re-derived from independent fixed-count calls, the
tile-wise ICD from the numpy implementation of tests/test_oracle_icd_pins.py extended by the stop rule.
"""
import numpy as np
import pytest

import smre_inputs as si

C = lambda sides: si.thresholds(sides).astype(np.float64)


# ---- standard variant ----------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,sides,delta", [(16, 19, [1, 2, 3], 1e-4), (21, 17, [2, 4], 1e-6), (12, 12, [3, 1, 5], 1e-2)])
def test_std_tol_stops_at_the_first_sweep_below_delta(oracle, H, W, sides, delta):
    """The returned sweep count r is the FIRST sweep with ||x_r - x_{r-1}||^2 <= delta, and x is the iterate
    after exactly r sweeps: both re-derived from fixed-count runs (which have their own pins)."""
    rng = np.random.default_rng(H + W)
    y = 2.0 * rng.standard_normal((H, W))
    c = C(sides)
    x, r = oracle.project_std_tol(y, sides, c, 2000, delta)
    assert 1 < r < 2000
    assert np.array_equal(x, oracle.project_std(y, sides, c, r))
    prev = y
    for k in range(1, r + 1):
        xk = oracle.project_std(y, sides, c, k)
        d2 = float(((xk - prev) ** 2).sum())
        assert (d2 <= delta) == (k == r), (k, r, d2)
        prev = xk


def test_std_tol_degenerate_cases(oracle):
    rng = np.random.default_rng(7)
    sides = [1, 2, 3, 4]
    c = C(sides)
    # feasible input: the first sweep changes nothing -> r = 1, x == y bit for bit (P2)
    y = 0.2 * rng.standard_normal((20, 23))
    x, r = oracle.project_std_tol(y, sides, c, 50, 1e-12)
    assert r == 1 and np.array_equal(x, y)
    # delta = 0 on an infeasible input never stops early: exactly max_sweeps, the fixed-count iterate
    y = 2.0 * rng.standard_normal((14, 15))
    x, r = oracle.project_std_tol(y, sides, c, 9, 0.0)
    assert r == 9 and np.array_equal(x, oracle.project_std(y, sides, c, 9))
    # a huge delta stops after the first sweep
    x, r = oracle.project_std_tol(y, sides, c, 9, 1e30)
    assert r == 1 and np.array_equal(x, oracle.project_std(y, sides, c, 1))
    # the stop sweep does not increase with delta
    rs = [oracle.project_std_tol(y, sides, c, 5000, d)[1] for d in (1e-10, 1e-8, 1e-6, 1e-4, 1e-2, 1.0)]
    assert all(a >= b for a, b in zip(rs, rs[1:])) and rs[0] > rs[-1]


def test_std_tol_approaches_the_projection(oracle):
    """As delta -> 0 the stopped iterate approaches the limit (the projection): the distance to a
    10^5-sweep iterate shrinks with delta."""
    rng = np.random.default_rng(3)
    y = 2.0 * rng.standard_normal((6, 6))
    sides, c = [1, 2, 3], C([1, 2, 3])
    lim = oracle.project_std(y, sides, c, 100000)
    err = [float(np.abs(oracle.project_std_tol(y, sides, c, 100000, d)[0] - lim).max()) for d in (1e-4, 1e-8, 1e-12)]
    assert err[0] > err[1] > err[2] and err[2] < 1e-4


# ---- incomplete variant --------------------------------------------------------------------------------
def tilewise_icd_tol(y, K, level_c, max_cycles, tol):
    """Listing 3 with its while loop: each virtual L x L tile of shift i iterates its nested levels K..i until the
    tile's sum of |e_old - e_new| over one cycle is <= tol * L^2, at most max_cycles cycles."""
    H, W = y.shape
    L = 1 << K
    x = y.astype(np.float64).copy()
    total, cmax = 0, 0
    for i in range(K + 1):
        org = ((1 << i) % L) - L
        for ty in range(org, H, L):
            for tx in range(org, W, L):
                if ty + L <= 0 or tx + L <= 0:
                    continue
                q = np.zeros((K + 1, L, L))
                cyc = 0
                while True:
                    delta = 0.0
                    for k in range(K, i - 1, -1):
                        s = 1 << k
                        for ly in range(0, L, s):
                            for lx in range(0, L, s):
                                gy, gx = ty + ly, tx + lx
                                if gy < 0 or gx < 0 or gy + s > H or gx + s > W:
                                    continue
                                old = x[gy:gy + s, gx:gx + s].copy()
                                v = old + q[k, ly:ly + s, lx:lx + s]
                                n2 = (v * v).sum()
                                xn = v * np.sqrt(level_c[k] / n2) if n2 > level_c[k] else v
                                q[k, ly:ly + s, lx:lx + s] = v - xn
                                x[gy:gy + s, gx:gx + s] = xn
                                delta += np.abs(old - xn).sum()
                    cyc += 1
                    if not (delta > tol * L * L) or cyc >= max_cycles:
                        break
                total += cyc
                cmax = max(cmax, cyc)
    return x, total, cmax


@pytest.mark.parametrize("H,W,K,tol", [(24, 24, 3, 1e-3), (19, 27, 2, 1e-2), (37, 33, 4, 1e-3), (8, 8, 3, 1e-4)])
def test_icd_tol_equals_tilewise_with_stop_rule(oracle, H, W, K, tol):
    rng = np.random.default_rng(220 + K)
    y = 2.0 * rng.standard_normal((H, W))
    sides = [1 << k for k in range(K + 1)]
    x, total, cmax = oracle.project_icd_tol(y, sides, C(sides), 400, tol)
    want, wtotal, wmax = tilewise_icd_tol(y, K, C(sides), 400, tol)
    np.testing.assert_allclose(x, want, rtol=0, atol=1e-12)
    assert (total, cmax) == (wtotal, wmax) and 1 < cmax < 400


def test_icd_tol_degenerate_cases(oracle):
    rng = np.random.default_rng(9)
    sides = [1, 2, 4, 8]
    c = C(sides)
    y = 2.0 * rng.standard_normal((26, 31))
    # with tol < 0 nothing stops early: the fixed-count ICD, exactly
    x, total, cmax = oracle.project_icd_tol(y, sides, c, 7, -1.0)
    assert cmax == 7 and np.array_equal(x, oracle.project_icd(y, sides, c, 7))
    # feasible input: every tile of every shift runs exactly one cycle and nothing changes
    yf = 0.2 * rng.standard_normal((26, 31))
    x, total, cmax = oracle.project_icd_tol(yf, sides, c, 50, 1e-3)
    tiles = sum(len([t for t in range(((1 << i) % 8) - 8, 26, 8) if t + 8 > 0]) *
                len([t for t in range(((1 << i) % 8) - 8, 31, 8) if t + 8 > 0]) for i in range(4))
    assert cmax == 1 and total == tiles and np.array_equal(x, yf)
    # the cycle counts do not increase with tol
    tots = [oracle.project_icd_tol(y, sides, c, 2000, t)[1] for t in (1e-6, 1e-4, 1e-2, 1.0)]
    assert all(a >= b for a, b in zip(tots, tots[1:])) and tots[0] > tots[-1]


# ---- per-tile counts and the replay used to check the kernel's fp32 stop decisions ---------------------
def test_icd_replay_of_own_counts_is_exact_and_detects_wrong_counts(oracle):
    rng = np.random.default_rng(31)
    y = 2.0 * rng.standard_normal((29, 42))
    sides = [1, 2, 4, 8]
    c = C(sides)
    x, total, cmax = oracle.project_icd_tol(y, sides, c, 300, 1e-3)
    x2, counts = oracle.project_icd_tol_counts(y, sides, c, 300, 1e-3)
    assert np.array_equal(x, x2)
    assert [t.shape for t in counts] == oracle.icd_tile_grid(29, 42, 3)
    assert sum(int(t.sum()) for t in counts) == total and max(int(t.max()) for t in counts) == cmax
    # the counts of the independent numpy tile-wise solve (same enumeration: shifts, then tile rows, then columns)
    want, wtotal, wmax = tilewise_icd_tol(y, 3, c, 300, 1e-3)
    assert (total, cmax) == (wtotal, wmax)
    # replaying its own decisions reproduces the result and finds nothing to object to, even with a zero band
    xr, bad = oracle.replay_icd(y, sides, c, 300, 1e-3, counts, 0.0)
    assert bad == 0 and np.array_equal(xr, x)
    # one cycle too few / too many on a tile that iterated: the deltas do not allow it
    i, (ty, tx) = max(((i, np.unravel_index(t.argmax(), t.shape)) for i, t in enumerate(counts)),
                      key=lambda a: counts[a[0]][a[1]])
    for d in (-1, +1):
        wrong = [t.copy() for t in counts]
        wrong[i][ty, tx] += d
        _, bad = oracle.replay_icd(y, sides, c, 300, 1e-3, wrong, 1e-6)
        assert bad == 1
