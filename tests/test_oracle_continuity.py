"""Pins of the oracle's local depth-continuity filter (the third filter; reading Q25).
Everything here runs without a GPU; the expected values come from the paper's / SPEC.md's statement of the rule,
from hand-enumerated cases and from an independent numpy formulation (shifted arrays instead of window loops)."""
import numpy as np
import pytest

import oracle

OK, NO_PLANE, CONTINUITY, MASKED = 0, 1, 5, 4


def _numpy_continuity(depth, window, gamma, delta):
    """independent formulation: one shifted copy of the padded map per window offset"""
    H, W = depth.shape
    hw = window // 2
    pad = np.zeros((H + 2 * hw, W + 2 * hw))
    pad[hw:hw + H, hw:hw + W] = depth
    count = np.zeros((H, W), int)
    for dy in range(-hw, hw + 1):
        for dx in range(-hw, hw + 1):
            if dx == 0 and dy == 0:
                continue
            nb = pad[hw + dy:hw + dy + H, hw + dx:hw + dx + W]
            count += ((nb > 0) & (np.abs(nb - depth) < gamma)).astype(int)
    keep = (depth > 0) & ~(count / float(window * window - 1) < delta)
    return np.where(keep, depth, 0.0), count


def test_constant_map_is_unchanged_spec_example():
    # SPEC.md:284 "constant-depth map, gamma=0.5 m, delta=0.3 -> unchanged" (also at the borders: a corner pixel of a
    # 5x5 window still has 8 of 24 consistent neighbours = 0.333 >= 0.3)
    d = np.full((12, 17), 7.25)
    out, reason = oracle.filter_continuity(d, 5, 0.5, 0.3)
    assert np.array_equal(out, d) and (reason == OK).all()


def test_isolated_spike_is_removed_spec_example():
    # SPEC.md:285 "isolated 50 m spike in a 10 m plane -> spike invalidated"; its neighbours keep 23 of 24
    d = np.full((11, 11), 10.0)
    d[5, 5] = 50.0
    out, reason = oracle.filter_continuity(d, 5, 0.5, 0.3)
    assert out[5, 5] == 0.0 and reason[5, 5] == CONTINUITY
    out[5, 5] = 10.0
    assert np.array_equal(out, np.full((11, 11), 10.0))


@pytest.mark.parametrize("k,kept", [(6, True), (5, False), (7, True)])
def test_exactly_delta_is_kept_hand_enumerated(k, kept):
    # SPEC.md:286 "exactly delta fraction consistent -> kept (strict less-than removes)": delta = 6/24 = 0.25
    d = np.zeros((5, 5))
    d[2, 2] = 4.0
    cells = [(0, 0), (0, 4), (4, 0), (4, 4), (1, 2), (2, 0), (3, 3)][:k]
    for (y, x) in cells:
        d[y, x] = 4.3  # |4.3 - 4.0| < 0.5
    d[2, 3] = 4.5      # |4.5 - 4.0| = 0.5 is NOT smaller than gamma: inconsistent
    d[0, 2] = 9.0      # valid but far
    out, reason = oracle.filter_continuity(d, 5, 0.5, 0.25)
    assert (out[2, 2] == 4.0) == kept
    assert reason[2, 2] == (OK if kept else CONTINUITY)


def test_invalid_neighbours_and_image_border_count_as_inconsistent():
    d = np.full((5, 5), 3.0)
    out, _ = oracle.filter_continuity(d, 5, 0.5, 0.3)
    assert out[0, 0] == 3.0            # 8/24 >= 0.3
    out, _ = oracle.filter_continuity(d, 5, 0.5, 0.34)
    assert out[0, 0] == 0.0            # 8/24 < 0.34: the 16 cells outside the image are not consistent
    assert out[2, 2] == 3.0            # 24/24
    d2 = d.copy()
    d2[0:2, :] = 0.0                   # invalid rows: centre keeps 14 of 24
    out, reason = oracle.filter_continuity(d2, 5, 0.5, 0.6)
    assert out[2, 2] == 0.0 and reason[2, 2] == CONTINUITY and reason[0, 0] == NO_PLANE
    out, _ = oracle.filter_continuity(d2, 5, 0.5, 14.0 / 24.0)
    assert out[2, 2] == 3.0


def test_reads_only_the_input_map_not_partially_filtered_state():
    # a ramp of pixels that would fall one after the other if the filter ran in place, row-major
    d = np.zeros((1, 9))
    d[0, :] = [1.0, 1.4, 1.8, 2.2, 2.6, 3.0, 3.4, 3.8, 4.2]
    out, _ = oracle.filter_continuity(d, 3, 0.5, 0.125)  # keep iff at least 1 of 8 consistent
    assert (out > 0).all()  # every pixel has a consistent horizontal neighbour in the INPUT


def test_matches_independent_numpy_formulation_and_is_contractive():
    rng = np.random.default_rng(5)
    for window, gamma, delta in ((5, 0.5, 0.3), (3, 0.25, 0.5), (7, 1.0, 0.2)):
        d = np.round(rng.uniform(2.0, 6.0, size=(37, 53)), 1)
        d[rng.uniform(size=d.shape) < 0.3] = 0.0
        ref, count = _numpy_continuity(d, window, gamma, delta)
        out, reason = oracle.filter_continuity(d, window, gamma, delta)
        assert np.array_equal(out, ref)
        assert ((out > 0) <= (d > 0)).all() and (out[out > 0] == d[out > 0]).all()  # contractive, values untouched
        assert ((reason == NO_PLANE) == (d == 0)).all()
        assert (reason[(d > 0) & (out == 0)] == CONTINUITY).all()
        assert 0 < (reason == CONTINUITY).sum() < (d > 0).sum()


def test_mask_is_applied_after_the_continuity_test():
    d = np.full((7, 7), 5.0)
    mask = np.zeros((7, 7), np.uint8)
    mask[3, :] = 1
    out, reason = oracle.filter_continuity(d, 5, 0.5, 0.3, mask)
    assert (out[3, :] == 0).all() and (reason[3, :] == MASKED).all()
    assert (out[[0, 1, 2, 4, 5, 6], :] == 5.0).all()  # masked neighbours still count: the mask comes last
    d[3, 3] = 50.0
    _, reason = oracle.filter_continuity(d, 5, 0.5, 0.3, mask)
    assert reason[3, 3] == CONTINUITY  # the continuity verdict wins over the mask


def test_window_must_be_odd():
    with pytest.raises(ValueError):
        oracle.filter_continuity(np.ones((4, 4)), 4, 0.5, 0.3)
