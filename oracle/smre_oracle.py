"""ctypes front end of oracle/smre_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
leg may import this module.  It never imports paper_1503_03492_b200 and shares
nothing with the CUDA path.

Every function takes float32 or float64 numpy arrays, up-casts them to float64
(readings A10: the fp32 threshold *values* are up-cast, so both sides compare
against numerically identical thresholds) and returns float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "smre_oracle.c")
_LIB = os.path.join(_HERE, "libsmre_oracle.so")

# Flags are part of the timed CPU baseline: -O2, no fast-math.
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    """Compile smre_oracle.c with gcc into oracle/libsmre_oracle.so."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        subprocess.check_call(["gcc", *CFLAGS, "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.smre_oracle_dykstra_families.restype = ctypes.c_int
        lib.smre_oracle_dykstra_families.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, _ip, _ip, _ip, _dp, ctypes.c_int,
            ctypes.c_int, _dp, _dp, ctypes.POINTER(ctypes.c_longlong)]
        lib.smre_oracle_std.restype = ctypes.c_int
        lib.smre_oracle_std.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, _ip, _dp, ctypes.c_int, ctypes.c_int,
            _dp, _dp, ctypes.POINTER(ctypes.c_longlong)]
        lib.smre_oracle_std_family_count.restype = ctypes.c_int
        lib.smre_oracle_std_family_count.argtypes = [_ip, ctypes.c_int]
        lib.smre_oracle_std_family_list.restype = None
        lib.smre_oracle_std_family_list.argtypes = [_ip, _dp, ctypes.c_int, _ip, _ip, _ip, _dp]
        lib.smre_oracle_icd_levels.restype = ctypes.c_int
        lib.smre_oracle_icd_levels.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, ctypes.c_int, _dp]
        lib.smre_oracle_icd.restype = ctypes.c_int
        lib.smre_oracle_icd.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, _ip, _dp, ctypes.c_int, ctypes.c_int, _dp]
        lib.smre_oracle_std_tol.restype = ctypes.c_int
        lib.smre_oracle_std_tol.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, _ip, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            _dp, _ip]
        lib.smre_oracle_icd_tol.restype = ctypes.c_int
        lib.smre_oracle_icd_tol.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, _ip, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            _dp, ctypes.POINTER(ctypes.c_longlong), _ip]
        lib.smre_oracle_icd_tiles_along.restype = ctypes.c_int
        lib.smre_oracle_icd_tiles_along.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.smre_oracle_icd_levels_tol_counts.restype = ctypes.c_int
        lib.smre_oracle_icd_levels_tol_counts.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, ctypes.c_int, ctypes.c_double, _dp, _ip]
        lib.smre_oracle_icd_levels_replay.restype = ctypes.c_int
        lib.smre_oracle_icd_levels_replay.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, ctypes.c_int, ctypes.c_double, _ip,
            ctypes.c_double, _dp, ctypes.POINTER(ctypes.c_longlong)]
        lib.smre_oracle_q_stat.restype = ctypes.c_int
        lib.smre_oracle_q_stat.argtypes = [_dp, ctypes.c_int, ctypes.c_int, _ip, ctypes.c_int, _dp]
        lib.smre_oracle_thresholds_from_q.restype = ctypes.c_int
        lib.smre_oracle_thresholds_from_q.argtypes = [_dp, ctypes.c_int, ctypes.c_double, _ip, ctypes.c_int, _dp, _dp]
        lib.smre_oracle_cumulant2.restype = ctypes.c_int
        lib.smre_oracle_cumulant2.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp]
        lib.smre_oracle_window_sums.restype = ctypes.c_int
        lib.smre_oracle_window_sums.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp]
        lib.smre_oracle_gauss_conv.restype = ctypes.c_int
        lib.smre_oracle_gauss_conv.argtypes = [_dp, ctypes.c_int, ctypes.c_int, ctypes.c_double, _dp]
        lib.smre_oracle_gauss_taps.restype = ctypes.c_int
        lib.smre_oracle_gauss_taps.argtypes = [ctypes.c_double, _dp, ctypes.c_int]
        lib.smre_oracle_admm.restype = ctypes.c_int
        lib.smre_oracle_admm.argtypes = [
            _dp, ctypes.c_int, ctypes.c_int, _ip, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int] + [ctypes.c_double] * 8 + [
            ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _ip, _dp]
        _lib = lib
    return _lib


def _f64(a):
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(np.asarray(a), dtype=np.int32)


def _p(a, t):
    return a.ctypes.data_as(t)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"{what} failed with code {rc}")


def std_family_list(sides, c):
    """Canonical ordered family list [(side, oy, ox, c)] of the exact method (A3)."""
    lib = _load()
    sides = _i32(sides)
    c = _f64(c)
    F = lib.smre_oracle_std_family_count(_p(sides, _ip), len(sides))
    fs, fy, fx = (np.zeros(F, np.int32) for _ in range(3))
    fc = np.zeros(F, np.float64)
    lib.smre_oracle_std_family_list(_p(sides, _ip), _p(c, _dp), len(sides),
                                    _p(fs, _ip), _p(fy, _ip), _p(fx, _ip), _p(fc, _dp))
    return [(int(a), int(b), int(d), float(e)) for a, b, d, e in zip(fs, fy, fx, fc)]


def dykstra_families(y, families, n_sweeps, return_q=False, return_active=False):
    """Cyclic Dykstra (Alg. 2) over an explicit ordered list [(side, oy, ox, c)]."""
    lib = _load()
    y = _f64(y)
    assert y.ndim == 2
    H, W = y.shape
    F = len(families)
    fs = _i32([f[0] for f in families])
    fy = _i32([f[1] for f in families])
    fx = _i32([f[2] for f in families])
    fc = _f64([f[3] for f in families])
    x = np.empty_like(y)
    q = np.zeros((F, H, W), np.float64) if return_q else None
    act = ctypes.c_longlong(0)
    rc = lib.smre_oracle_dykstra_families(
        _p(y, _dp), H, W, _p(fs, _ip), _p(fy, _ip), _p(fx, _ip), _p(fc, _dp), F,
        int(n_sweeps), _p(x, _dp), _p(q, _dp) if return_q else None, ctypes.byref(act))
    _check(rc, "smre_oracle_dykstra_families")
    out = (x,)
    if return_q:
        out += (q,)
    if return_active:
        out += (act.value,)
    return out if len(out) > 1 else x


def project_std(y, sides, c, n_sweeps, return_q=False):
    """Algorithm O-STD on one image [H,W] or a stack [B,H,W] (frames independent)."""
    lib = _load()
    y = _f64(y)
    sides = _i32(sides)
    c = _f64(c)
    if y.ndim == 3:
        res = [project_std(f, sides, c, n_sweeps, return_q) for f in y]
        if return_q:
            return np.stack([r[0] for r in res]), np.stack([r[1] for r in res], axis=1)
        return np.stack(res)
    H, W = y.shape
    x = np.empty_like(y)
    q = None
    if return_q:
        F = lib.smre_oracle_std_family_count(_p(sides, _ip), len(sides))
        q = np.zeros((F, H, W), np.float64)
    rc = lib.smre_oracle_std(_p(y, _dp), H, W, _p(sides, _ip), _p(c, _dp), len(sides),
                             int(n_sweeps), _p(x, _dp), _p(q, _dp) if return_q else None, None)
    _check(rc, "smre_oracle_std")
    return (x, q) if return_q else x


def project_icd(y, sides, c, n_sweeps):
    """Algorithm O-ICD on one image [H,W] or a stack [B,H,W] (frames independent)."""
    lib = _load()
    y = _f64(y)
    sides = _i32(sides)
    c = _f64(c)
    if y.ndim == 3:
        return np.stack([project_icd(f, sides, c, n_sweeps) for f in y])
    H, W = y.shape
    x = np.empty_like(y)
    rc = lib.smre_oracle_icd(_p(y, _dp), H, W, _p(sides, _ip), _p(c, _dp), len(sides),
                             int(n_sweeps), _p(x, _dp))
    _check(rc, "smre_oracle_icd")
    return x


def project_std_tol(y, sides, c, max_sweeps, delta):
    """Alg. 2 with its stop rule ||x_r - x_{r-1}||^2 <= delta per sweep.
    One image [H,W] -> (x, sweeps_done); a stack [B,H,W] -> (x, [sweeps_done per frame])."""
    lib = _load()
    y = _f64(y)
    sides = _i32(sides)
    c = _f64(c)
    if y.ndim == 3:
        res = [project_std_tol(f, sides, c, max_sweeps, delta) for f in y]
        return np.stack([r[0] for r in res]), [r[1] for r in res]
    H, W = y.shape
    x = np.empty_like(y)
    done = ctypes.c_int(0)
    rc = lib.smre_oracle_std_tol(_p(y, _dp), H, W, _p(sides, _ip), _p(c, _dp), len(sides),
                                 int(max_sweeps), float(delta), _p(x, _dp), ctypes.byref(done))
    _check(rc, "smre_oracle_std_tol")
    return x, done.value


def project_icd_tol(y, sides, c, max_cycles, tol):
    """Incomplete variant, every tile iterated until Listing 3's sum |delta| <= tol * L^2.
    One image [H,W] -> (x, cycles_total, cycles_max); a stack -> (x, sum, max) over the frames."""
    lib = _load()
    y = _f64(y)
    sides = _i32(sides)
    c = _f64(c)
    if y.ndim == 3:
        res = [project_icd_tol(f, sides, c, max_cycles, tol) for f in y]
        return np.stack([r[0] for r in res]), sum(r[1] for r in res), max(r[2] for r in res)
    H, W = y.shape
    x = np.empty_like(y)
    tot, mx = ctypes.c_longlong(0), ctypes.c_int(0)
    rc = lib.smre_oracle_icd_tol(_p(y, _dp), H, W, _p(sides, _ip), _p(c, _dp), len(sides),
                                 int(max_cycles), float(tol), _p(x, _dp), ctypes.byref(tot), ctypes.byref(mx))
    _check(rc, "smre_oracle_icd_tol")
    return x, tot.value, mx.value


def _icd_levels(sides, c):
    sides = [int(v) for v in sides]
    K = int(np.floor(np.log2(max(sides))))
    c_of = {s: float(v) for s, v in zip(sides, c)}
    return K, _f64([c_of[1 << k] for k in range(K + 1)])


def icd_tile_grid(H, W, K):
    """[(tiles along y, tiles along x)] per shift i = 0..K: the layout of the per-tile cycle counts."""
    lib = _load()
    return [(lib.smre_oracle_icd_tiles_along(int(H), K, i), lib.smre_oracle_icd_tiles_along(int(W), K, i))
            for i in range(K + 1)]


def project_icd_tol_counts(y, sides, c, max_cycles, tol):
    """As project_icd_tol on ONE image, returning (x, [per shift: int32 array (ty, tx) of cycles run])."""
    lib = _load()
    y = _f64(y)
    H, W = y.shape
    K, lc = _icd_levels(sides, c)
    grid = icd_tile_grid(H, W, K)
    counts = np.zeros(sum(a * b for a, b in grid), np.int32)
    x = np.empty_like(y)
    _check(lib.smre_oracle_icd_levels_tol_counts(_p(y, _dp), H, W, K, _p(lc, _dp), int(max_cycles), float(tol),
                                                 _p(x, _dp), _p(counts, _ip)), "smre_oracle_icd_levels_tol_counts")
    out, o = [], 0
    for a, b in grid:
        out.append(counts[o:o + a * b].reshape(a, b).copy())
        o += a * b
    return x, out


def replay_icd(y, sides, c, max_cycles, tol, tile_cycles, band):
    """Every tile runs exactly the cycles tile_cycles prescribes (list per shift of (ty, tx) arrays, e.g. the CUDA
    path's); returns (x, n_bad): n_bad tiles whose count the fp64 deltas do not allow within the relative band."""
    lib = _load()
    y = _f64(y)
    H, W = y.shape
    K, lc = _icd_levels(sides, c)
    grid = icd_tile_grid(H, W, K)
    assert len(tile_cycles) == K + 1 and all(np.asarray(t).shape == g for t, g in zip(tile_cycles, grid))
    counts = _i32(np.concatenate([np.asarray(t).ravel() for t in tile_cycles]))
    x = np.empty_like(y)
    bad = ctypes.c_longlong(0)
    _check(lib.smre_oracle_icd_levels_replay(_p(y, _dp), H, W, K, _p(lc, _dp), int(max_cycles), float(tol),
                                             _p(counts, _ip), float(band), _p(x, _dp), ctypes.byref(bad)),
           "smre_oracle_icd_levels_replay")
    return x, bad.value


def q_stat(eps, sides):
    """Q_Omega of one image [H,W], or of every frame of a stack [n,H,W] -> array [n]."""
    lib = _load()
    eps = _f64(eps)
    sides = _i32(sides)
    if eps.ndim == 3:
        return np.array([q_stat(f, sides) for f in eps])
    H, W = eps.shape
    q = ctypes.c_double(0.0)
    _check(lib.smre_oracle_q_stat(_p(eps, _dp), H, W, _p(sides, _ip), len(sides), ctypes.byref(q)), "smre_oracle_q_stat")
    return q.value


def thresholds_from_q(q, alpha, sides):
    """(q_alpha, thresholds c_S = (q_alpha sigma_s + mu_s)^4 per side) from simulated Q values."""
    lib = _load()
    q = _f64(q).ravel()
    sides = _i32(sides)
    c = np.zeros(len(sides), np.float64)
    qa = ctypes.c_double(0.0)
    _check(lib.smre_oracle_thresholds_from_q(_p(q, _dp), len(q), float(alpha), _p(sides, _ip), len(sides),
                                             ctypes.byref(qa), _p(c, _dp)), "smre_oracle_thresholds_from_q")
    return qa.value, c


def cumulant2(stack):
    """C_2(r, 0) = <F^2>_t - <F>_t^2 per pixel of a stack [n,H,W] (Eq. 19)."""
    lib = _load()
    stack = _f64(stack)
    n, H, W = stack.shape
    out = np.empty((H, W), np.float64)
    _check(lib.smre_oracle_cumulant2(_p(stack, _dp), n, H, W, _p(out, _dp)), "smre_oracle_cumulant2")
    return out


def gauss_taps(sigma):
    """Normalised taps of the Gaussian PSF, radius ceil(3 sigma) (reading A-ADMM-2)."""
    lib = _load()
    t = np.zeros(257, np.float64)
    r = lib.smre_oracle_gauss_taps(float(sigma), _p(t, _dp), 257)
    if r < 0:
        raise RuntimeError("smre_oracle_gauss_taps failed")
    return t[:2 * r + 1].copy()


def gauss_conv(x, sigma):
    """A * x: separable Gaussian of standard deviation sigma, zero outside the image (= A^T * x)."""
    lib = _load()
    x = _f64(x)
    H, W = x.shape
    out = np.empty((H, W), np.float64)
    _check(lib.smre_oracle_gauss_conv(_p(x, _dp), H, W, float(sigma), _p(out, _dp)), "smre_oracle_gauss_conv")
    return out


def admm(I, sides, c, variant, n_sweeps, sigma, rho1, rho2, alpha1, alpha2, lam, gamma, delta, max_iter):
    """Alg. 1 with the z = x splitting (smre_oracle.c has the update rules and the readings).
    Returns a dict: x, eps, z, Y1, Y2, iters, hist[iters, 2] = (||x_r - x_{r-1}||, ||I - A x_r - eps_r||)."""
    lib = _load()
    I = _f64(I)
    H, W = I.shape
    sides = _i32(sides)
    c = _f64(c)
    outs = [np.empty((H, W), np.float64) for _ in range(5)]
    it = np.zeros(1, np.int32)
    hist = np.zeros(2 * int(max_iter), np.float64)
    v = 0 if variant in ("standard", 0) else 1
    _check(lib.smre_oracle_admm(_p(I, _dp), H, W, _p(sides, _ip), _p(c, _dp), len(sides), v, int(n_sweeps),
                                float(sigma), float(rho1), float(rho2), float(alpha1), float(alpha2), float(lam),
                                float(gamma), float(delta), int(max_iter), *[_p(o, _dp) for o in outs],
                                _p(it, _ip), _p(hist, _dp)), "smre_oracle_admm")
    n = int(it[0])
    return dict(x=outs[0], eps=outs[1], z=outs[2], Y1=outs[3], Y2=outs[4], iters=n, hist=hist[:2 * n].reshape(n, 2))


def project(y, sides, c, n_sweeps, variant):
    if variant in ("standard", 0):
        return project_std(y, sides, c, n_sweeps)
    if variant in ("incomplete", 1):
        return project_icd(y, sides, c, n_sweeps)
    raise ValueError(variant)


def window_sums(x, s):
    """t_s of every s x s window fully inside the image, all shifts: [(H-s+1),(W-s+1)]."""
    lib = _load()
    x = _f64(x)
    H, W = x.shape
    out = np.empty((H - s + 1, W - s + 1), np.float64)
    _check(lib.smre_oracle_window_sums(_p(x, _dp), H, W, int(s), _p(out, _dp)),
           "smre_oracle_window_sums")
    return out
