"""Parity protocol between the CUDA path and the fp64 oracle (BASELINE.json north_star;
SURVEY.md 8(c) "GPU-vs-oracle parity protocol").  Test infrastructure only.

  * max |x_gpu - x_ref| <= 1e-4 * max|y|   over all pixels and frames
  * the set of violated windows (t_S > c_S, evaluated in fp64 on either output) must agree
    exactly, except windows within 1e-5 relative of c_S in either output.
    Window collection: standard -> every window of every side at every shift;
    incomplete -> the windows of its own level passes (reading A-ICD-7/14).
"""
import numpy as np

import smre_inputs as si

TOL_REL = 1e-4
BAND = 1e-5


def _ratios(oracle, x, sides, c, variant):
    """List of fp64 arrays t_S / c_S, one per window collection entry."""
    out = []
    if variant == "standard":
        for s, cs in zip(sides, c):
            out.append(oracle.window_sums(x, int(s)) / float(cs))
    else:
        K = int(np.floor(np.log2(max(int(s) for s in sides))))
        c_of = {int(s): float(cs) for s, cs in zip(sides, c)}
        sums = {}
        for (_, _, side, o) in si.icd_level_passes(K):
            if side not in sums:
                sums[side] = oracle.window_sums(x, side)
            out.append(sums[side][o::side, o::side] / c_of[side])
    return out


def compare(oracle, y, x_gpu, x_ref, sides, c, variant):
    """Returns a dict of diagnostics; raises AssertionError when the protocol is violated."""
    y = np.asarray(y)
    x_gpu = np.asarray(x_gpu, dtype=np.float64).reshape(y.shape)
    x_ref = np.asarray(x_ref, dtype=np.float64).reshape(y.shape)
    tol = TOL_REL * float(np.abs(y).max())
    err = float(np.abs(x_gpu - x_ref).max())
    assert np.isfinite(x_gpu).all()
    assert err <= tol, f"max|x_gpu - x_ref| = {err:.3e} > {tol:.3e}"
    frames_g = x_gpu.reshape(-1, y.shape[-2], y.shape[-1])
    frames_r = x_ref.reshape(-1, y.shape[-2], y.shape[-1])
    n_viol = n_band = n_win = 0
    for fg, fr in zip(frames_g, frames_r):
        for rg, rr in zip(_ratios(oracle, fg, sides, c, variant), _ratios(oracle, fr, sides, c, variant)):
            band = (np.abs(rg - 1.0) <= BAND) | (np.abs(rr - 1.0) <= BAND)
            vg, vr = (rg > 1.0) & ~band, (rr > 1.0) & ~band
            assert np.array_equal(vg, vr), (
                f"violated-window sets differ on {int((vg != vr).sum())} windows "
                f"(worst ratio gpu {rg.max():.8f}, ref {rr.max():.8f})")
            n_viol += int(vr.sum())
            n_band += int(band.sum())
            n_win += rg.size
    return {"max_abs_err": err, "tol": tol, "violated": n_viol, "in_band": n_band, "windows": n_win}
