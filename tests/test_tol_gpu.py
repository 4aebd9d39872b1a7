"""GPU parity of the convergence-controlled projection (smre_project_tol) against the oracle's stop-rule modes.

The stop decision compares a floating-point sum with a threshold, so the fp32 kernel and the fp64 oracle may
legitimately stop a borderline sweep / tile one iteration apart ("a parity rule tolerant of +-1").
The protocol used here is stricter than +-1: the kernel's OWN counts are checked against the fp64 quantities within a
relative band (every earlier iteration must have been above the threshold, the last one below it), and the image is
compared, at the usual tolerance, with the oracle run for exactly those counts.
"""
import numpy as np
import pytest

import smre_inputs as si
from tests import parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1503_03492_b200 as smre  # noqa: E402

BAND = 1e-4            # relative band around the threshold inside which either decision is accepted


def check_std_decision(oracle, y, sides, c, delta, r_gpu, max_sweeps):
    """r_gpu must be a legitimate stop sweep of Alg. 2 within the band."""
    prev = np.asarray(y, np.float64)
    for k in range(1, r_gpu + 1):
        xk = oracle.project_std(y, sides, c, k)
        d2 = float(((xk - prev) ** 2).sum())
        if k < r_gpu:
            assert d2 > delta * (1 - BAND), (k, r_gpu, d2)
        elif r_gpu < max_sweeps:
            assert d2 <= delta * (1 + BAND), (k, r_gpu, d2)
        prev = xk
    return prev


@pytest.mark.parametrize("idx,delta,max_sweeps", [(0, 1e-3, 500), (0, 1e-1, 500), (0, 1e-9, 25), (1, 0.5, 60)])
def test_standard_stops_where_alg2_says(oracle, idx, delta, max_sweeps):
    w = si.config(idx)
    sol = smre.Solver(w.H, w.W, w.sides, w.c, "standard")
    x, done = sol.project_tol(torch.from_numpy(w.y).cuda(), max_sweeps, delta)
    torch.cuda.synchronize()
    r_gpu = int(done.cpu()[0])
    assert sol.last_launch[0] == smre.SMRE_SCHED_STRIPS
    _, r_ref = oracle.project_std_tol(w.y, w.sides, w.c, max_sweeps, delta)
    print(f"\n{w.name} delta={delta}: sweeps gpu {r_gpu}, oracle {r_ref}")
    assert abs(r_gpu - r_ref) <= 1 and 1 <= r_gpu <= max_sweeps
    x_ref = check_std_decision(oracle, w.y, w.sides, w.c, delta, r_gpu, max_sweeps)
    parity.compare(oracle, w.y, x.cpu().numpy(), x_ref, w.sides, w.c, "standard")
    # the same call again stops on the same sweep with the same bits; a fixed-count call gives them too
    x2, done2 = sol.project_tol(torch.from_numpy(w.y).cuda(), max_sweeps, delta)
    assert int(done2.cpu()[0]) == r_gpu and torch.equal(x, x2)
    assert torch.equal(sol.project(torch.from_numpy(w.y).cuda(), r_gpu), x)
    sol.close()


def test_standard_batch_frames_stop_on_their_own(oracle):
    rng = np.random.default_rng(8)
    sides = [1, 2, 3, 4]
    c = si.thresholds(sides)
    y = np.stack([0.2 * rng.standard_normal((70, 90)),            # feasible: stops after sweep 1, returned bit for bit
                  1.8 * rng.standard_normal((70, 90)),
                  1.2 * rng.standard_normal((70, 90))]).astype(np.float32)
    sol = smre.Solver(70, 90, sides, c, "standard", batch=3)
    x, done = sol.project_tol(torch.from_numpy(y).cuda(), 300, 1e-4)
    torch.cuda.synchronize()
    done = done.cpu().numpy()
    assert done[0] == 1 and np.array_equal(x.cpu().numpy()[0], y[0])
    assert done[1] > done[2] > 1
    for b in range(3):
        x_ref = check_std_decision(oracle, y[b], sides, c, 1e-4, int(done[b]), 300)
        parity.compare(oracle, y[b], x.cpu().numpy()[b], x_ref, sides, c, "standard")
    sol.close()


@pytest.mark.parametrize("idx,tol,max_cycles", [(2, 1e-3, 2000), (4, 1e-3, 2000), (3, 1e-3, 2000)])
def test_incomplete_tiles_stop_where_listing3_says(oracle, idx, tol, max_cycles):
    w = si.config(idx)
    frames = w.y if w.y.ndim == 3 else w.y[None]
    if frames.shape[0] > 4:
        frames = frames[:4]                                       # C4: four frames keep the oracle replay short
    sol = smre.Solver(w.H, w.W, w.sides, w.c, "incomplete", batch=frames.shape[0])
    x, done = sol.project_tol(torch.from_numpy(np.ascontiguousarray(frames)).cuda(), max_cycles, tol)
    cycles = [t.cpu().numpy() for t in sol.tile_cycles()]
    torch.cuda.synchronize()
    x = x.cpu().numpy()
    assert int(done.cpu()[0]) == max(int(t.max()) for t in cycles)
    total_gpu = sum(int(t.sum()) for t in cycles)
    total_ref = 0
    for b in range(frames.shape[0]):
        # the kernel's counts are legitimate stop decisions of Listing 3, and the image is what those counts give
        x_ref, bad = oracle.replay_icd(frames[b], w.sides, w.c, max_cycles, tol, [t[b] for t in cycles], BAND)
        assert bad == 0
        parity.compare(oracle, frames[b], x[b], x_ref, w.sides, w.c, "incomplete")
        _, tot, _ = oracle.project_icd_tol(frames[b], w.sides, w.c, max_cycles, tol)
        total_ref += tot
    print(f"\n{w.name} tol={tol}: tile cycles gpu {total_gpu}, oracle {total_ref}, max {int(done.cpu()[0])}")
    assert abs(total_gpu - total_ref) <= 1e-3 * total_ref + 2
    # early exit pays: far fewer cycles than the fixed-count configuration runs
    n_tiles = sum(t.size for t in cycles)
    assert total_gpu < 0.8 * n_tiles * w.n_sweeps
    sol.close()


def test_tol_degenerate_and_errors(oracle):
    rng = np.random.default_rng(2)
    sides = [1, 2, 4, 8]
    c = si.thresholds(sides)
    yf = (0.2 * rng.standard_normal((40, 56))).astype(np.float32)      # feasible
    for variant in ("standard", "incomplete"):
        sol = smre.Solver(40, 56, sides, c, variant)
        x, done = sol.project_tol(torch.from_numpy(yf).cuda(), 50, 1e-3)
        assert int(done.cpu()[0]) == 1 and np.array_equal(x.cpu().numpy(), yf)
        with pytest.raises(smre.SmreError) as e:
            smre.smre_project_tol(sol.handle, x.data_ptr(), x.data_ptr(), 0, 1e-3)
        assert e.value.status == smre.smre.SMRE_EINVAL
        with pytest.raises(smre.SmreError):
            smre.smre_project_tol(sol.handle, x.data_ptr(), x.data_ptr(), 5, -1.0)
        sol.close()
    # tol = 0 on an infeasible image: the fixed-count result of max_sweeps
    y = (1.8 * rng.standard_normal((40, 56))).astype(np.float32)
    sol = smre.Solver(40, 56, sides, c, "standard")
    x, done = sol.project_tol(torch.from_numpy(y).cuda(), 9, 0.0)
    assert int(done.cpu()[0]) == 9 and torch.equal(x, sol.project(torch.from_numpy(y).cuda(), 9))
    sol.close()
