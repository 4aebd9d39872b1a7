"""Host logic of the conveyor scheduler (no GPU): the planner tiles the bench workload onto <= 148 CTAs and
every hand-off invariant holds for every step (smre_plan_check runs the planner's own verifier)."""
import pytest

import paper_1503_03492_b200 as smre


def test_c1_plan_fits_one_cta_per_sm():
    ty, tx, mh, mw, tb = smre.smre_plan_check(512, 512, range(1, 9), 6)
    assert ty * tx <= 148 and ty >= 8 and tx >= 8
    assert mh <= 56 and mw <= 56                      # tile + two steps of movement fit the 64-entry torus
    assert tb == 204 * 6 * (ty + tx) * 16


def test_small_images_are_one_static_tile():
    assert smre.smre_plan_check(64, 64, [1, 2, 3, 4], 50)[:4] == (1, 1, 64, 64)
    assert smre.smre_plan_check(37, 53, [1, 2, 3, 4, 5], 7)[:2] == (1, 1)


@pytest.mark.parametrize("H,W,sides,n", [(100, 300, [1, 2, 3, 4, 5], 6), (256, 256, list(range(1, 9)), 4),
                                          (40, 72, [16, 5], 4), (200, 90, [3, 1, 6], 5)])
def test_ragged_plans_verify(H, W, sides, n):
    ty, tx, mh, mw, _ = smre.smre_plan_check(H, W, sides, n)
    assert ty * tx <= 148 and mh <= 64 and mw <= 64


def test_too_large_for_one_wave_is_refused():
    with pytest.raises(smre.SmreError) as e:
        smre.smre_plan_check(1024, 1024, range(1, 9), 2)
    assert e.value.status == smre.smre.SMRE_EUNSUPPORTED
    assert "CTAs" in str(e.value)
    # more CTAs allowed -> a plan exists
    ty, tx, *_ = smre.smre_plan_check(1024, 1024, range(1, 9), 2, max_ctas=1024)
    assert ty * tx > 148


def test_bad_arguments():
    for args in [(0, 8, [1], 1), (8, 8, [9], 1), (8, 8, [1], 0)]:
        with pytest.raises(smre.SmreError) as e:
            smre.smre_plan_check(*args)
        assert e.value.status == smre.smre.SMRE_EINVAL


def test_spare_slot_when_death_and_birth_touch():
    # 113 = 7 * 16 + 1: the one-row tile at the bottom dies in the step before the same slot would be born at the top
    ty, tx, *_ = smre.smre_plan_check(113, 88, [8, 7, 6, 5, 4, 3, 2, 1], 3)
    assert (ty, tx) == (9, 7)
