"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element,
on the five BASELINE.json configs at full size and on small / ragged / degenerate cases."""
import numpy as np
import pytest

import smre_inputs as si
from tests import parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
import paper_1503_03492_b200 as smre  # noqa: E402

SCHEDULES = {"graph": smre.SMRE_SCHED_GRAPH, "persistent": smre.SMRE_SCHED_PERSISTENT,
             "strips": smre.SMRE_SCHED_STRIPS}


def gpu_project(y, sides, c, variant, n_sweeps, schedule=smre.SMRE_SCHED_AUTO, in_place=False):
    y = np.ascontiguousarray(y, dtype=np.float32)
    batch = 1 if y.ndim == 2 else y.shape[0]
    sol = smre.Solver(y.shape[-2], y.shape[-1], sides, c, variant, batch, schedule)
    try:
        yt = torch.from_numpy(y).cuda()
        out = sol.project(yt, n_sweeps, out=yt if in_place else None)
        torch.cuda.synchronize()
        return out.cpu().numpy(), sol.last_launch
    finally:
        sol.close()


# ---- the five configs, full size, in the launch configuration bench.py times -------------------
@pytest.mark.parametrize("idx", [0, 1, 2, 3, 4])
def test_config_full_size(oracle, idx):
    w = si.config(idx)
    x_gpu, launch = gpu_project(w.y, w.sides, w.c, w.variant, w.n_sweeps)
    x_ref = oracle.project(w.y, w.sides, w.c, w.n_sweeps, w.variant)
    d = parity.compare(oracle, w.y, x_gpu, x_ref, w.sides, w.c, w.variant)
    print(f"\n{w.name}: {d} launch={launch}")
    assert d["violated"] + d["in_band"] > 0          # finite sweeps: the comparison is not vacuous
    assert launch[1] > 0


# ---- every scheduler of the standard variant gives the same bits -------------------------------
@pytest.mark.parametrize("idx,n", [(0, 50), (1, 3)])
def test_schedulers_agree_bitwise(idx, n):
    w = si.config(idx)
    res = {}
    for name, sch in SCHEDULES.items():
        try:
            res[name], launch = gpu_project(w.y, w.sides, w.c, "standard", n, sch)
            assert launch[0] == sch
        except smre.SmreError as e:
            assert e.status == smre.smre.SMRE_EUNSUPPORTED
    assert "graph" in res
    for name, x in res.items():
        assert np.array_equal(x, res["graph"]), name


# ---- the persistent schedulers are deterministic: repeated calls give the graph scheduler's bits every time ----
@pytest.mark.parametrize("sched", ["persistent", "strips"])
def test_persistent_repeatable(sched):
    for idx, n, reps in ((0, 20, 25), (1, 2, 6)):
        w = si.config(idx)
        ref, _ = gpu_project(w.y, w.sides, w.c, "standard", n, smre.SMRE_SCHED_GRAPH)
        sol = smre.Solver(w.H, w.W, w.sides, w.c, "standard", 1, SCHEDULES[sched])
        yt = torch.from_numpy(w.y).cuda()
        for _ in range(reps):
            x = sol.project(yt, n)
            torch.cuda.synchronize()
            assert sol.last_launch[0] == SCHEDULES[sched]
            assert np.array_equal(x.cpu().numpy(), ref)
        sol.close()


# ---- several tiles, short sweeps: q written by one CTA is read a sweep later by another one ------------------
@pytest.mark.parametrize("H,W,B,sides,n", [(160, 176, 2, [1, 2, 3, 4], 4), (128, 128, 1, [1, 2, 3, 4], 5),
                                           (200, 200, 1, [1, 2, 3, 4, 5, 6], 3), (256, 256, 2, list(range(1, 9)), 2),
                                           (96, 300, 1, [2, 3, 5], 4),
                                           # a tile row / column that dies at the far edge one step before the same CTA
                                           # slot would host the newborn one at the near edge (needs the spare slot)
                                           (113, 88, 1, [8, 7, 6, 5, 4, 3, 2, 1], 3), (160, 175, 1, [6, 8, 3], 3),
                                           (407, 71, 2, [1, 2, 3, 4, 5, 6, 7], 3), (384, 97, 1, [4, 5, 6, 7, 8], 3),
                                           # q ordering across sweeps: many narrow tiles and a short sweep (a pixel changes
                                           # owner six times per sweep; window grids that nest, so boundaries often rest and
                                           # carry no hand-off), chains of empty slots
                                           (492, 54, 1, [2, 4, 6, 8], 3), (98, 437, 2, [1, 2, 4, 8], 4),
                                           (142, 553, 2, [1, 2, 4, 8], 2), (187, 447, 3, [1, 2, 4, 8], 3)])
def test_persistent_schedulers_match_graph_bitwise(H, W, B, sides, n):
    """Both persistent schedulers against one kernel per family, bit for bit.  The strips take every one of these
    shapes; the conveyor refuses multi-tile problems whose sweep is shorter than its ordering margin (F < ~40) --
    that refusal is asserted, not skipped, and SMRE_SCHED_AUTO must still run such a problem persistently."""
    rng = np.random.default_rng(H + W)
    y = (1.6 * rng.standard_normal((B, H, W))).astype(np.float32)
    y[:, : H // 2, : W // 2] += 1.5
    c = si.thresholds(sides)
    ref, _ = gpu_project(y, sides, c, "standard", n, smre.SMRE_SCHED_GRAPH)
    for _ in range(2):
        x, launch = gpu_project(y, sides, c, "standard", n, smre.SMRE_SCHED_STRIPS)
        assert launch[0] == smre.SMRE_SCHED_STRIPS and launch[2] > 1
        assert np.array_equal(x, ref)
    F = sum(s * s for s in sides)
    try:
        x, launch = gpu_project(y, sides, c, "standard", n, smre.SMRE_SCHED_PERSISTENT)
        assert launch[2] * launch[3] > 1
        assert np.array_equal(x, ref)
    except smre.SmreError as e:
        assert e.status == smre.smre.SMRE_EUNSUPPORTED and F < 64, (F, str(e))
    x, launch = gpu_project(y, sides, c, "standard", n, smre.SMRE_SCHED_AUTO)
    assert launch[0] in (smre.SMRE_SCHED_PERSISTENT, smre.SMRE_SCHED_STRIPS)
    assert np.array_equal(x, ref)


def test_conveyor_random_shapes_match_graph_bitwise():
    rng = np.random.default_rng(2024)
    pools = [list(range(1, 9)), list(range(1, 7)), [2, 3, 5, 7], [1, 3, 5, 6, 8], [4, 5, 6, 7, 8], [8, 7, 6, 5, 4, 3, 2, 1]]
    ran = 0
    for _ in range(40):
        H, W = int(rng.integers(65, 420)), int(rng.integers(65, 420))
        B, n = int(rng.integers(1, 3)), int(rng.integers(2, 4))
        sides = pools[int(rng.integers(len(pools)))]
        y = (1.6 * rng.standard_normal((B, H, W))).astype(np.float32)
        y[:, : H // 2, : W // 2] += 1.5
        c = si.thresholds(sides)
        try:
            x, launch = gpu_project(y, sides, c, "standard", n, smre.SMRE_SCHED_PERSISTENT)
        except smre.SmreError as e:
            assert e.status == smre.smre.SMRE_EUNSUPPORTED, (H, W, B, sides, n, str(e))
            continue
        ref, _ = gpu_project(y, sides, c, "standard", n, smre.SMRE_SCHED_GRAPH)
        assert np.array_equal(x, ref), (H, W, B, sides, n, launch)
        xs, ls = gpu_project(y, sides, c, "standard", n, smre.SMRE_SCHED_STRIPS)
        assert np.array_equal(xs, ref), (H, W, B, sides, n, ls)
        ran += 1
        if ran >= 12:
            break
    assert ran >= 6


# ---- small, ragged, degenerate --------------------------------------------------------------------
CASES = [
    # H, W, batch, sides, variant, sweeps
    (37, 53, 1, [1, 2, 3, 4, 5], "standard", 7),          # ragged: nothing divides
    (64, 40, 3, [3, 1, 6], "standard", 5),                # batch > 1, sides not ascending
    (33, 35, 1, [7, 8], "standard", 9),
    (40, 72, 2, [16, 5], "standard", 4),
    (70, 66, 1, [32, 17, 2], "standard", 3),              # largest compiled side
    (160, 176, 2, [1, 2, 3, 4], "standard", 4),           # F = 30: graph and strips (40 strips x 2 frames); the conveyor refuses
    (8, 8, 1, [8], "standard", 3),                        # one window = the image
    (5, 7, 1, [1], "standard", 2),                        # clip only
    (50, 61, 1, [1, 2, 4, 8], "incomplete", 11),          # ragged ICD, K = 3
    (64, 64, 5, [1, 2, 3, 4, 5, 6, 7, 8], "incomplete", 20),
    (45, 99, 2, [1, 2, 4, 8, 16], "incomplete", 6),       # K = 4
    (70, 83, 2, [1, 2, 4, 8, 16, 32], "incomplete", 5),   # K = 5, the paper's own depth
    (19, 23, 1, [1, 2, 4], "incomplete", 8),              # K = 2
    (9, 11, 3, [1, 2], "incomplete", 4),                  # K = 1
    (6, 5, 1, [1], "incomplete", 3),                      # K = 0
    (16, 16, 1, [1, 2, 4, 8, 16], "incomplete", 9),       # image = one tile
]


@pytest.mark.parametrize("H,W,B,sides,variant,n", CASES)
def test_small_and_ragged(oracle, H, W, B, sides, variant, n):
    rng = np.random.default_rng(H * 1000 + W)
    y = (1.6 * rng.standard_normal((B, H, W))).astype(np.float32)
    y[:, : H // 2, : W // 2] += 1.5
    if B == 1:
        y = y[0]
    c = si.thresholds(sides)
    x_ref = oracle.project(y, sides, c, n, variant)
    scheds = list(SCHEDULES.values()) if variant == "standard" else [smre.SMRE_SCHED_AUTO]
    ran = 0
    for sch in scheds:
        try:
            x_gpu, _ = gpu_project(y, sides, c, variant, n, sch)
        except smre.SmreError as e:
            assert e.status == smre.smre.SMRE_EUNSUPPORTED and sch != smre.SMRE_SCHED_GRAPH
            continue
        ran += 1
        d = parity.compare(oracle, y, x_gpu, x_ref, sides, c, variant)
        assert np.abs(x_ref - y).max() > 0.05, "vacuous case"
        assert d["max_abs_err"] < 2e-5
    assert ran >= 1


def test_in_place_and_identity_on_feasible_input(oracle):
    rng = np.random.default_rng(5)
    sides = np.arange(1, 9)
    c = si.thresholds(sides)
    y = (0.2 * rng.standard_normal((48, 52))).astype(np.float32)       # feasible: P2
    for variant in ("standard", "incomplete"):
        x, _ = gpu_project(y, sides, c, variant, 3)
        assert np.array_equal(x, y)
    w = si.config(0)
    for variant in ("standard", "incomplete"):
        a, _ = gpu_project(w.y, [1, 2, 4], si.thresholds([1, 2, 4]), variant, 6)
        b, _ = gpu_project(w.y, [1, 2, 4], si.thresholds([1, 2, 4]), variant, 6, in_place=True)
        assert np.array_equal(a, b)
    # in place under each scheduler of the standard variant, several strips / tiles
    w1 = si.config(1)
    a, _ = gpu_project(w1.y, w1.sides, w1.c, "standard", 2, smre.SMRE_SCHED_GRAPH)
    for sch in SCHEDULES.values():
        b, launch = gpu_project(w1.y, w1.sides, w1.c, "standard", 2, sch, in_place=True)
        assert launch[0] == sch and np.array_equal(a, b)


def test_exported_increments_and_host_path(oracle):
    w = si.config(0)
    sol = smre.Solver(w.H, w.W, w.sides, w.c, "standard")
    yt = torch.from_numpy(w.y).cuda()
    x = sol.project(yt, 20)
    q = sol.increments()
    torch.cuda.synchronize()
    x_ref, q_ref = oracle.project_std(w.y, w.sides, w.c, 20, return_q=True)
    assert sol.info == (30, 15630, 30 * 64 * 64 * 4)
    fams = oracle.std_family_list(w.sides, w.c)
    for i, f in enumerate(sol.families()):
        assert f[:3] == fams[i][:3] and abs(f[3] - fams[i][3]) < 1e-6
    qn = q.cpu().numpy()[:, 0].astype(np.float64)
    # conservation x + sum_f q_f == y (P5) holds on the GPU too, up to fp32 rounding
    assert np.abs(x.cpu().numpy() + qn.sum(0) - w.y).max() < 2e-5
    assert np.abs(qn - q_ref).max() < 2e-5
    # same windows carry a multiplier, away from the decision boundary
    big = np.abs(q_ref) > 1e-4
    assert np.array_equal(np.abs(qn) > 0, np.abs(q_ref) > 0) or (np.abs(qn)[big] > 0).all()
    # a second call starts from q = 0 again (no state carried between calls)
    x2 = sol.project(yt, 20)
    assert torch.equal(x, x2)
    xh = sol.project_host(w.y, 20)
    assert np.array_equal(xh, x.cpu().numpy())
    sol.close()


@pytest.mark.parametrize("sched", ["persistent", "strips"])
def test_increments_of_pixels_outside_every_window_are_zero(oracle, sched):
    """q of pixels no window of a family covers (rows < oy, columns < ox, remainders) must read 0 after a call of a
    persistent scheduler, whatever the allocation held before: they are zeroed at create and never written."""
    H, W, sides, n = 67, 70, [3, 5, 2], 6
    c = si.thresholds(sides)
    F = sum(s * s for s in sides)
    dirty = torch.full((F * H * ((W + 3) // 4 * 4) + 1024,), 7.25, device="cuda")   # same size as the q planes
    torch.cuda.synchronize()
    del dirty                                                   # the caching allocator hands the block out again
    rng = np.random.default_rng(3)
    y = (1.8 * rng.standard_normal((H, W))).astype(np.float32)
    sol = smre.Solver(H, W, sides, c, "standard", 1, SCHEDULES[sched])
    x = sol.project(torch.from_numpy(y).cuda(), n)
    q = sol.increments().cpu().numpy()[:, 0].astype(np.float64)
    torch.cuda.synchronize()
    assert sol.last_launch[0] == SCHEDULES[sched]
    x_ref, q_ref = oracle.project_std(y, sides, c, n, return_q=True)
    assert np.abs(q - q_ref).max() < 2e-5
    for i, (s, oy, ox, _) in enumerate(sol.families()):
        cov = np.zeros((H, W), bool)
        cov[oy:oy + (H - oy) // s * s, ox:ox + (W - ox) // s * s] = True
        assert (q[i][~cov] == 0).all(), (i, s, oy, ox)
    assert np.abs(x.cpu().numpy() + q.sum(0) - y).max() < 2e-5          # conservation (P5)
    sol.close()


def test_error_codes_on_device():
    sol = smre.Solver(16, 16, [1, 2], si.thresholds([1, 2]), "standard")
    yt = torch.zeros(16, 16, device="cuda")
    with pytest.raises(smre.SmreError) as e:
        smre.smre_project(sol.handle, yt.data_ptr(), yt.data_ptr(), 0, 0)
    assert e.value.status == smre.smre.SMRE_EINVAL
    with pytest.raises(smre.SmreError):
        smre.smre_project(sol.handle, None, yt.data_ptr(), 1, 0)
    with pytest.raises(smre.SmreError):
        smre.smre_family(sol.handle, 99)
    sol.close()
    with pytest.raises(smre.SmreError) as e:
        smre.Solver(16, 16, [1, 2, 8], si.thresholds([1, 2, 8]), "incomplete")   # level 4 missing
    assert e.value.status == smre.smre.SMRE_EINVAL
    icd = smre.Solver(16, 16, [1, 2], si.thresholds([1, 2]), "incomplete")
    assert icd.info[0] == 3 and icd.info[2] == 0
    with pytest.raises(smre.SmreError):
        icd.increments()
    icd.close()
