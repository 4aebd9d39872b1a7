"""Pins of the oracle's incomplete-Dykstra (ICD) function and of the counting helpers (CPU only).

PAPER.md sec. 3.2 (365-395) + Listing 2/3.  The ICD is a heuristic with no closed-form
target, so it is pinned by (a) an explicit block-local, tile-by-tile solve written here in
the shape of Listing 3 (one 2^K x 2^K tile at a time, local q[level] arrays, levels coarse to
fine), (b) its decomposition into standard Dykstra runs on restricted family lists, and
(c) its degenerate cases.
"""
import numpy as np
import pytest

import smre_inputs as si

C = lambda sides: si.thresholds(sides).astype(np.float64)


def tilewise_icd(y, K, level_c, n_cycles):
    """Listing 3 shaped reference: for each shift i (Listing 2), for each virtual L x L tile
    with origin (2^i - L + m L) on both axes, run the block-local Dykstra over the nested levels
    K..i with tile-local q, skipping windows that are not fully inside the image (A-ICD-13)."""
    H, W = y.shape
    L = 1 << K
    x = y.astype(np.float64).copy()
    for i in range(K + 1):
        org = ((1 << i) % L) - L if ((1 << i) % L) else 0
        for ty in range(org, H, L):
            for tx in range(org, W, L):
                q = np.zeros((K + 1, L, L))                       # "Set q = 0"
                for _ in range(n_cycles):
                    for k in range(K, i - 1, -1):                 # for (s = 5; s >= smin; s--)
                        s = 1 << k
                        for ly in range(0, L, s):
                            for lx in range(0, L, s):
                                gy, gx = ty + ly, tx + lx
                                if gy < 0 or gx < 0 or gy + s > H or gx + s > W:
                                    continue
                                v = x[gy:gy + s, gx:gx + s] + q[k, ly:ly + s, lx:lx + s]
                                n2 = (v * v).sum()
                                xn = v * np.sqrt(level_c[k] / n2) if n2 > level_c[k] else v
                                q[k, ly:ly + s, lx:lx + s] = v - xn
                                x[gy:gy + s, gx:gx + s] = xn
    return x


# ---- P12a: ICD == explicit tile-by-tile block-local solve -------------------------------------
@pytest.mark.parametrize("H,W,K,n", [(24, 24, 3, 6), (19, 27, 2, 5), (37, 33, 4, 3), (8, 8, 3, 9)])
def test_icd_equals_tilewise(oracle, H, W, K, n):
    rng = np.random.default_rng(120 + K)
    y = 2.0 * rng.standard_normal((H, W))
    sides = [1 << k for k in range(K + 1)]
    x = oracle.project_icd(y, sides, C(sides), n)
    want = tilewise_icd(y, K, C(sides), n)
    np.testing.assert_allclose(x, want, rtol=0, atol=1e-13)
    assert np.abs(x - y).max() > 0.1                              # the case is not vacuous


# ---- P12b: ICD == S_K o ... o S_0, S_i = standard Dykstra from q = 0 on [(2^k, o, o)]_k=K..i ---
@pytest.mark.parametrize("K", [2, 3, 4])
def test_icd_is_composition_of_restricted_standard_runs(oracle, K):
    rng = np.random.default_rng(12)
    y = 2.0 * rng.standard_normal((45, 52))
    sides = [1 << k for k in range(K + 1)]
    c = C(sides)
    x = y
    n_pass = 0
    for i in range(K + 1):
        fams = [((1 << k), (1 << i) % (1 << k), (1 << i) % (1 << k), float(c[k])) for k in range(K, i - 1, -1)]
        n_pass += len(fams)
        x = oracle.dykstra_families(x, fams, 7)
    assert n_pass == {2: 6, 3: 10, 4: 15}[K]
    assert np.array_equal(oracle.project_icd(y, sides, c, 7), x)


def test_icd_ignores_non_power_of_two_sides_and_needs_all_levels(oracle):
    rng = np.random.default_rng(13)
    y = 2.0 * rng.standard_normal((32, 32))
    a = oracle.project_icd(y, np.arange(1, 9), C(np.arange(1, 9)), 4)        # sides 1..8 -> K = 3
    b = oracle.project_icd(y, [1, 2, 4, 8], C([1, 2, 4, 8]), 4)
    assert np.array_equal(a, b)
    with pytest.raises(RuntimeError):
        oracle.project_icd(y, [1, 2, 8], C([1, 2, 8]), 4)                    # level 4 missing


# ---- P13: the last shift i = K is one exact projection onto the un-shifted L-tiling -----------
def test_icd_last_shift_feasible_on_unshifted_tiles(oracle):
    w = si.config(0)
    sides = [1, 2, 4, 8]
    c = C(sides)
    x = oracle.project_icd(w.y, sides, c, 30)
    t = oracle.window_sums(x, 8)[::8, ::8]
    assert t.max() <= c[3] * (1 + 1e-12)
    # side-1 windows are only visited in shift 0, yet stay feasible: later steps only shrink |x_i|
    assert np.abs(x).max() <= np.sqrt(c[0]) * (1 + 1e-12)


# ---- P14: degenerate cases -----------------------------------------------------------------------
def test_icd_degenerate_cases(oracle):
    rng = np.random.default_rng(14)
    y = 3.0 * rng.standard_normal((16, 16))
    # image = one L x L tile, only level L constrained in effect (other thresholds huge) -> Eq. 14
    sides, c = [1, 2, 4, 8, 16], np.array([1e9, 1e9, 1e9, 1e9, 100.0])
    x = oracle.project_icd(y, sides, c, 3)
    np.testing.assert_allclose(x, y * np.sqrt(100.0 / (y * y).sum()), rtol=1e-14)
    # n_sweeps = 1: plain cyclic projections, no increment is ever re-used
    sides = [1, 2, 4]
    cc = C(sides)
    x1 = oracle.project_icd(y, sides, cc, 1)
    z = y.copy()
    for i in range(3):
        for k in range(2, i - 1, -1):
            s, o = 1 << k, (1 << i) % (1 << k)
            for wy in range(o, 16 - s + 1, s):
                for wx in range(o, 16 - s + 1, s):
                    b = z[wy:wy + s, wx:wx + s]
                    n2 = (b * b).sum()
                    if n2 > cc[k]:
                        z[wy:wy + s, wx:wx + s] = b * np.sqrt(cc[k] / n2)
    np.testing.assert_allclose(x1, z, rtol=1e-15)


# ---- P15: counts (BASELINE.json configs) -----------------------------
def test_counts(oracle):
    assert [si.std_family_count(range(1, n + 1)) for n in (4, 8, 16)] == [30, 204, 1496]
    assert len(oracle.std_family_list(np.arange(1, 9), C(np.arange(1, 9)))) == 204
    assert si.std_windows_per_sweep(64, 64, range(1, 5)) == 15630
    assert si.std_windows_per_sweep(512, 512, range(1, 9)) == 2068620
    assert si.std_windows_per_sweep(1024, 1024, range(1, 17)) == 16532696
    assert 64 * si.std_windows_per_sweep(256, 256, range(1, 9)) == 32645888
    assert [len(si.icd_level_passes(K)) for K in (3, 4, 5)] == [10, 15, 21]
    assert si.icd_level_passes(3) == [(0, 3, 8, 1), (0, 2, 4, 1), (0, 1, 2, 1), (0, 0, 1, 0),
                                      (1, 3, 8, 2), (1, 2, 4, 2), (1, 1, 2, 0),
                                      (2, 3, 8, 4), (2, 2, 4, 0), (3, 3, 8, 0)]
    assert si.icd_windows_per_cycle(512, 512, 3) == 457350
    assert si.icd_windows_per_cycle(1024, 1024, 4) == 1852170
    assert 64 * si.icd_windows_per_cycle(256, 256, 3) == 7295360
    # the windows the oracle really visits in one standard sweep == the formula (border rule A6)
    fams = oracle.std_family_list([1, 2, 3, 4], C([1, 2, 3, 4]))
    n = sum(((64 - oy) // s) * ((64 - ox) // s) for s, oy, ox, _ in fams)
    assert n == 15630


# ---- P16: the paper's storage figures ---------------------------------------
def test_storage_figures():
    assert 15 ** 3 * 1024 ** 2 * 4 == 14155776000                 # "14 GB", O(L^3 L_I^2) literally
    assert (6 + 2) * 4 == 32 and 3 * 4 == 12                      # ICD 32 B/thread, exact 12 B/thread
    assert si.std_family_count(range(1, 9)) * 512 * 512 * 4 == 213909504   # C1 q planes, 204 MiB


# ---- generators are deterministic and have the stated shapes ----------------------------------
def test_input_generators_seeded():
    a, b = si.config(0), si.config(0)
    assert np.array_equal(a.y, b.y) and a.y.dtype == np.float32 and a.y.shape == (64, 64)
    w1, w2 = si.config(1), si.config(2)
    assert np.array_equal(w1.y, w2.y) and w1.y.shape == (512, 512)
    assert w1.variant == "standard" and w2.variant == "incomplete" and w1.n_sweeps == 200
    s = si.sofi_stack(B=3, H=32, W=32)
    assert s.shape == (3, 32, 32) and not np.array_equal(s[0], s[1])
    p = si.poisson_image(H=64, W=64, n_spots=10)
    assert abs(p.std() - 1.0) < 0.1 and abs(p.mean()) < 0.1
