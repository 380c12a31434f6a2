"""The numpy bank model of the scatter kernel (tests/bank_model.py) held to the two ncu measurements there are and to the
figures DESIGN.md §5 quotes from it -- `-m "not gpu"`; a model of ONE resource (shared-memory wavefronts per ATOMS), not a
timing."""
import numpy as np
import pytest

import bank_model as bm


@pytest.fixture(scope="module")
def samples():
    return bm.Samples(trials=1500, seed=1)


def test_model_reproduces_both_ncu_measurements(samples):
    """profiles/README.md (round 1, r1_scatter_full.csv): 2.96 wavefronts per ATOMS for the 16 x 2 layout, 4.17 for the
    forward kernel's 8 x 4 layout without skew"""
    lm1 = bm.score(samples, *bm.LAYOUTS["LM1 16x2, rows 8 apart (ncu: 2.96)"])[0]
    plain84 = bm.score(samples, *bm.LAYOUTS["8x4 without skew (ncu: 4.17)"])[0]
    assert abs(lm1 - 2.96) <= 0.04 * 2.96 and abs(plain84 - 4.17) <= 0.04 * 4.17, (lm1, plain84)


def test_shipped_layout_and_the_floor_of_any_rearrangement(samples):
    plain, merged, same = bm.score(samples, *bm.LAYOUTS["LM0 8x4, two-sample skew per row (shipped)"])
    assert abs(plain - 2.23) <= 0.08 and abs(merged - 2.01) <= 0.08 and 0.40 <= same <= 0.48, (plain, merged, same)   # tests/cpu_shim: 2.25 / 2.01
    best = bm.search(samples, skews=(0, 2))
    assert best[0][1] == 32 and 1.70 <= best[0][0] <= 1.85, best[:3]        # 32 pixels of one detector row per warp, row pitch 0 mod 32
    assert merged <= 1.15 * best[0][0]                                      # the shipped layout is within ~12 % of the floor
    best16 = min(r for r in best if r[1] == 16)
    assert 1.85 <= best16[0] <= 1.98 and best16[3] == 16, best16            # the best layout that keeps the 16 x 16 tile
