"""Seeded synthetic workloads (BASELINE.json configs 0-4; recipe in DESIGN.md sec. 5).

This module serves BOTH the oracle and the CUDA path and therefore holds none of
the method's arithmetic: it only draws residual images and lists the window sides
and their thresholds.  The images stand in for the paper's test photograph with
noise sigma in {1,3,10} and its 3091-frame SOFI movie
(PAPER.md:535), neither of which is available.

Recipe: rng = numpy.random.default_rng(seed) (PCG64); draw order = noise field
first, then the spot parameters; everything is generated in float64 and cast once
to float32; both sides consume the same float32 array.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


def thresholds(sides) -> np.ndarray:
    """c_S = |S| + 2*sqrt(2|S|), |S| = side^2 (BASELINE.json configs; chi^2 mean + 2 std
    at sigma = 1), rounded once to float32 -- the table both sides receive."""
    n = np.asarray(sides, dtype=np.float64) ** 2
    return (n + 2.0 * np.sqrt(2.0 * n)).astype(np.float32)


@dataclass
class Workload:
    name: str
    y: np.ndarray                 # float32, [H,W] or [B,H,W]
    sides: np.ndarray             # int32
    c: np.ndarray                 # float32 thresholds, one per side
    variant: str                  # "standard" | "incomplete"
    n_sweeps: int
    note: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def batch(self) -> int:
        return 1 if self.y.ndim == 2 else self.y.shape[0]

    @property
    def H(self) -> int:
        return self.y.shape[-2]

    @property
    def W(self) -> int:
        return self.y.shape[-1]


def _gauss_spots(H, W, rows, cols, sigmas, amps):
    rr = np.arange(H, dtype=np.float64)[:, None]
    cc = np.arange(W, dtype=np.float64)[None, :]
    img = np.zeros((H, W), np.float64)
    for r0, c0, sg, a in zip(rows, cols, sigmas, amps):
        img += a * np.exp(-((rr - r0) ** 2 + (cc - c0) ** 2) / (2.0 * sg * sg))
    return img


def blobs_image(H=64, W=64, seed=0, n_blobs=3, blob=8, amp=4.0) -> np.ndarray:
    """configs[0]: N(0,1) + n_blobs square blobs of +amp at seeded integer origins."""
    rng = np.random.default_rng(seed)
    img = rng.standard_normal((H, W))
    oy = rng.integers(0, H - blob + 1, size=n_blobs)
    ox = rng.integers(0, W - blob + 1, size=n_blobs)
    for a, b in zip(oy, ox):
        img[a:a + blob, b:b + blob] += amp
    return img.astype(np.float32)


def spots_image(H=512, W=512, seed=1, n_spots=40, sigma=(1.0, 3.0), amp=(2.0, 6.0)) -> np.ndarray:
    """configs[1]/[2]: N(0,1) + Gaussian spots, sigma_px ~ U(sigma), amplitude ~ U(amp)."""
    rng = np.random.default_rng(seed)
    img = rng.standard_normal((H, W))
    rows = rng.uniform(0, H, n_spots)
    cols = rng.uniform(0, W, n_spots)
    sg = rng.uniform(sigma[0], sigma[1], n_spots)
    am = rng.uniform(amp[0], amp[1], n_spots)
    return (img + _gauss_spots(H, W, rows, cols, sg, am)).astype(np.float32)


def poisson_image(H=1024, W=1024, seed=3, n_spots=400, sigma=1.5) -> np.ndarray:
    """configs[3]: (Poisson(lam) - lam)/sqrt(lam), lam = 50 + 200*signal, signal = spots/max."""
    rng = np.random.default_rng(seed)
    rows = rng.uniform(0, H, n_spots)
    cols = rng.uniform(0, W, n_spots)
    sig = _gauss_spots(H, W, rows, cols, np.full(n_spots, sigma), np.ones(n_spots))
    sig /= sig.max()
    lam = 50.0 + 200.0 * sig
    counts = rng.poisson(lam).astype(np.float64)
    return ((counts - lam) / np.sqrt(lam)).astype(np.float32)


def sofi_stack(B=64, H=256, W=256, seed=4, n_spots=60, sigma=2.0, amp=(1.0, 5.0), jitter=0.5) -> np.ndarray:
    """configs[4]: B frames, N(0,1) + n_spots Gaussian emitters; base positions and
    amplitudes drawn once from `seed`, per-frame position jitter N(0, jitter px) and
    noise from default_rng(1000*seed + frame)."""
    base = np.random.default_rng(seed)
    rows = base.uniform(0, H, n_spots)
    cols = base.uniform(0, W, n_spots)
    am = base.uniform(amp[0], amp[1], n_spots)
    out = np.empty((B, H, W), np.float32)
    for f in range(B):
        rng = np.random.default_rng(1000 * seed + f)
        noise = rng.standard_normal((H, W))
        jr = rng.normal(0.0, jitter, n_spots)
        jc = rng.normal(0.0, jitter, n_spots)
        out[f] = (noise + _gauss_spots(H, W, rows + jr, cols + jc,
                                       np.full(n_spots, sigma), am)).astype(np.float32)
    return out


def _sides(lo, hi):
    return np.arange(lo, hi + 1, dtype=np.int32)


def config(idx: int, n_sweeps: int | None = None) -> Workload:
    """BASELINE.json configs[idx]."""
    if idx == 0:
        s = _sides(1, 4)
        w = Workload("C0_64_std", blobs_image(), s, thresholds(s), "standard", 50,
                     "64x64 N(0,1)+3 blobs, sides 1-4, standard, 50 sweeps")
    elif idx == 1:
        s = _sides(1, 8)
        w = Workload("C1_512_std", spots_image(), s, thresholds(s), "standard", 200,
                     "512x512 N(0,1)+40 spots, sides 1-8 (204 families), standard, 200 sweeps")
    elif idx == 2:
        s = _sides(1, 8)
        w = Workload("C2_512_icd", spots_image(), s, thresholds(s), "incomplete", 200,
                     "same image as C1, incomplete Dykstra K=3, 200 inner cycles per shift")
    elif idx == 3:
        s = _sides(1, 16)
        w = Workload("C3_1024_icd", poisson_image(), s, thresholds(s), "incomplete", 100,
                     "1024x1024 Poisson residual, sides 1-16 -> K=4, 100 inner cycles per shift")
    elif idx == 4:
        s = _sides(1, 8)
        w = Workload("C4_64x256_icd", sofi_stack(), s, thresholds(s), "incomplete", 100,
                     "64 frames 256x256 SOFI-like, K=3, 100 inner cycles per shift, one call")
    else:
        raise ValueError(f"no config {idx}")
    if n_sweeps is not None:
        w.n_sweeps = int(n_sweeps)
    return w


def std_family_count(sides) -> int:
    return int(sum(int(s) * int(s) for s in sides))


def std_windows_per_sweep(H, W, sides) -> int:
    """sum_s (H-s+1)(W-s+1): every window of the exact method is visited once per sweep."""
    return int(sum((H - int(s) + 1) * (W - int(s) + 1) for s in sides))


def icd_level_passes(K):
    """[(shift i, level k, side, diagonal offset)] in execution order (Listing 2/3)."""
    out = []
    for i in range(K + 1):
        for k in range(K, i - 1, -1):
            side = 1 << k
            out.append((i, k, side, (1 << i) % side))
    return out


def icd_windows_per_cycle(H, W, K) -> int:
    n = 0
    for (_, _, side, o) in icd_level_passes(K):
        n += ((H - o) // side) * ((W - o) // side)
    return n
