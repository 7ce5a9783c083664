"""The hit-list comparison the GPU parity tests rely on (tests/gpu_helpers.compare_hits), checked on hand-made lists."""
import numpy as np

from gpu_helpers import compare_hits


def _h(rows):
    a = np.array(rows, dtype=np.int64).reshape(-1, 3)
    return a[:, 0], a[:, 1], a[:, 2]


def test_identical_lists():
    rows = [(5, 100, 80), (5, 140, 81), (9, 30, 200)]
    assert compare_hits(_h(rows), _h(rows)) == (1.0, True, 3, 3, 0)


def test_near_miss_takes_the_later_hits_of_the_pixel_with_it():
    orc = [(5, 100, 80), (5, 140, 81), (5, 190, 90), (9, 30, 200)]
    gpu = [(5, 100, 80), (5, 141, 81), (5, 193, 95), (9, 30, 200)]      # one tick late at the second crossing, then adrift
    frac, ok, ng, no, near = compare_hits(_h(gpu), _h(orc))
    assert ok and near == 1 and (ng, no) == (4, 4) and frac == 2 / 4


def test_one_count_at_a_code_boundary_does_not_excuse_what_follows():
    orc = [(5, 100, 80), (5, 140, 81), (5, 190, 90)]
    frac, ok, ng, no, near = compare_hits(_h([(5, 100, 80), (5, 140, 82), (5, 190, 90)]), _h(orc))
    assert ok and near == 1 and frac == 2 / 3
    assert not compare_hits(_h([(5, 100, 80), (5, 140, 82), (5, 193, 90)]), _h(orc))[1]    # later hit adrift: not excused


def test_first_difference_beyond_one_tick_or_count_fails():
    orc = [(5, 100, 80), (5, 140, 81)]
    assert not compare_hits(_h([(5, 100, 80), (5, 142, 81)]), _h(orc))[1]
    assert not compare_hits(_h([(5, 100, 82), (5, 140, 81)]), _h(orc))[1]


def test_missing_and_extra_hits_fail():
    orc = [(5, 100, 80), (5, 140, 81)]
    assert not compare_hits(_h([(5, 100, 80)]), _h(orc))[1]                       # a hit is missing
    assert not compare_hits(_h(orc + [(7, 10, 10)]), _h(orc))[1]                   # a pixel the oracle never fired
    assert not compare_hits(_h(orc), _h(orc + [(7, 10, 10)]))[1]
