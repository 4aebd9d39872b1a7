"""smre_project_noalloc (the entry point that allocates nothing, include/smre.h) against the existing path.

Collected last on purpose (the suite runs with pytest -x).  The new entry point keeps its increment planes in a
static device array that every call shares and that keeps the last call's contents, so the check runs on TWO calls
in a row with different inputs and sizes: the second one must not see anything of the first.
"""
import numpy as np
import pytest

import smre_inputs as si
from tests import parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1503_03492_b200 as smre  # noqa: E402


def existing_path(y, sides, c, n):
    sol = smre.Solver(y.shape[0], y.shape[1], sides, c, "standard", 1, smre.SMRE_SCHED_GRAPH)
    try:
        x = sol.project(torch.from_numpy(y).cuda(), n)
        torch.cuda.synchronize()
        return x.cpu().numpy()
    finally:
        sol.close()


def no_alloc_path(y, sides, c, n, in_place=False, check_free=False):
    yt = torch.from_numpy(y).cuda()
    out = yt if in_place else torch.empty_like(yt)
    st = torch.cuda.current_stream()
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]                 # cudaMemGetInfo: what the DRIVER has handed out
    smre.smre_project_noalloc(y.shape[0], y.shape[1], sides, c, yt.data_ptr(), out.data_ptr(), n, st.cuda_stream)
    torch.cuda.synchronize()
    if check_free:                                              # (not on the first call: kernels load lazily)
        assert torch.cuda.mem_get_info()[0] >= free_before
    return out.cpu().numpy()


def test_no_alloc_matches_existing_path_on_two_calls_in_a_row(oracle):
    w = si.config(0)                                            # 64 x 64, sides 1-4, 30 families
    rng = np.random.default_rng(11)
    y2 = (1.7 * rng.standard_normal((45, 83))).astype(np.float32)      # ragged, other sides: other plane layout
    y2[:20, :30] += 1.5
    sides2 = np.array([3, 1, 5], np.int32)
    c2 = si.thresholds(sides2)
    cases = [(w.y, w.sides, w.c, 12), (y2, sides2, c2, 7), (w.y, w.sides, w.c, 12)]
    for k, (y, sides, c, n) in enumerate(cases):
        x_new = no_alloc_path(y, sides, c, n, check_free=k == 2)
        x_old = existing_path(y, sides, c, n)
        tol = parity.TOL_REL * float(np.abs(y).max())
        assert np.abs(x_new - x_old).max() <= tol, k
        assert np.array_equal(x_new, x_old), k                  # same kernel, same order: the same bits
        d = parity.compare(oracle, y, x_new, oracle.project(y, sides, c, n, "standard"), sides, c, "standard")
        assert np.abs(x_new - y).max() > 0.05 and d["max_abs_err"] < 2e-5
    # in place
    assert np.array_equal(no_alloc_path(w.y, w.sides, w.c, 5, in_place=True), existing_path(w.y, w.sides, w.c, 5))


def test_no_alloc_rejects_what_does_not_fit():
    y = torch.zeros(1024, 1024, device="cuda")
    sides = np.arange(1, 9, dtype=np.int32)
    with pytest.raises(smre.SmreError) as e:
        smre.smre_project_noalloc(1024, 1024, sides, si.thresholds(sides), y.data_ptr(), y.data_ptr(), 1, 0)
    assert e.value.status == smre.smre.SMRE_EUNSUPPORTED and "SMRE_NOALLOC_MAX_BYTES" in str(e.value)
    with pytest.raises(smre.SmreError) as e:
        smre.smre_project_noalloc(16, 16, [1, 2], si.thresholds([1, 2]), None, y.data_ptr(), 1, 0)
    assert e.value.status == smre.smre.SMRE_EINVAL
