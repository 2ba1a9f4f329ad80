"""Host logic of the colour-class program generator (no GPU): which colour multisets are structurally non-zero,
and how the work is dealt over lanes.  The generator lives in libbg.so (csrc/bg_program.cpp); the expected
validity comes from the workload's colour rule g8, which tests/test_workload.py pins against the oracle."""
import itertools

import numpy as np
import pytest


@pytest.fixture(scope="module")
def bg():
    import paper_2106_06507_b200 as bg
    bg.load()
    return bg


def multisets(n):
    for comb in itertools.combinations_with_replacement(range(9), n):
        yield comb


@pytest.mark.parametrize("n", [4, 5, 6])
def test_class_validity_is_the_colour_rule(bg, wl, n):
    nvalid = 0
    for codes in multisets(n):
        counts = np.bincount(codes, minlength=9)
        valid = bg.bg_class_program_stats(n, 4, counts)[0]
        col = np.array([[c // 3 + 1, c % 3 + 1] for c in codes], dtype=np.int8)
        # rule g8 is invariant under relabelling the gluons, so it is a property of the multiset
        expect = wl.colour_valid(col)
        assert bool(valid) == bool(expect), (codes, valid, expect)
        nvalid += valid
    assert nvalid == {4: 21, 5: 45, 6: 92}[n]        # the distinct classes 65536 sampled events fall into


@pytest.mark.parametrize("n", [6, 8, 9])
def test_lane_schedules_cover_the_same_work(bg, wl, n):
    ev = wl.config_events(4, N=64, n=n)
    code = (ev.col[:, :, 0].astype(int) - 1) * 3 + (ev.col[:, :, 1].astype(int) - 1)
    for e in range(0, 64, 7):
        counts = np.bincount(code[e], minlength=9)
        ref = bg.bg_class_program_stats(n, 1, counts)
        assert ref[0] == 1 and ref[2] >= ref[1]            # one lane: every vertex is a step (plus setup steps)
        for lanes in (2, 4, 8, 32, 128):
            st = bg.bg_class_program_stats(n, lanes, counts)
            assert st[0] == 1
            assert st[1] == ref[1] or st[4] != ref[4]      # same vertices unless another closure leg was cheaper
            assert st[2] <= ref[2]                         # more lanes never need more steps
            assert st[2] * lanes >= st[1]                  # and cannot beat perfect balance


def test_bad_arguments(bg):
    with pytest.raises(bg.BgError):
        bg.bg_class_program_stats(6, 3, np.array([6, 0, 0, 0, 0, 0, 0, 0, 0]))
    with pytest.raises(bg.BgError):
        bg.bg_class_program_stats(6, 4, np.array([5, 0, 0, 0, 0, 0, 0, 0, 0]))


def connected_orderings(codes):
    """Brute force over the (n-1)! orderings of Eq. 19 with gluon 0 first: those whose deltas are all one."""
    n = len(codes)
    ci, cj = [c // 3 for c in codes], [c % 3 for c in codes]
    cnt = 0
    for rest in itertools.permutations(range(1, n)):
        o = (0,) + rest
        cnt += all(cj[o[k]] == ci[o[(k + 1) % n]] for k in range(n))
    return cnt


@pytest.mark.parametrize("n", [4, 5, 6])
def test_comc_programs_sum_the_colour_connected_orderings(bg, wl, oracle, n):
    mom = wl.config_events(4, N=1, n=n).mom
    hel = np.ones((1, n), dtype=np.int8)
    for codes in multisets(n):
        counts = np.bincount(codes, minlength=9)
        valid, nvert, steps, state, nord = bg.bg_comc_program_stats(n, 4, counts)
        expect = connected_orderings(codes)
        assert nord == expect and bool(valid) == (expect > 0), (codes, nord, expect)
        col = np.array([[[c // 3 + 1, c % 3 + 1] for c in codes]], dtype=np.int8)
        # rule g8 is stricter: e.g. all gluons in one U(1) colour state connect in every ordering but sum to zero
        assert bool(valid) or not wl.colour_valid(col[0])
        if valid:
            # the oracle's Eq. 19 brute force counts the same orderings
            assert oracle.colour_flow(mom, hel, col, return_count=True)[1][0] == nord
            # currents of shared sub-sequences are evaluated once: never more vertices than ordering-by-ordering
            per_ordering = sum((n - L) * (L - 1) for L in range(2, n))     # splits of all sub-sequences, Eq. 20
            assert 0 < nvert <= nord * per_ordering and steps * 4 >= nvert
    same = np.zeros(9, dtype=np.int64)
    same[0] = n
    assert bg.bg_comc_program_stats(n, 4, same)[4] == {4: 6, 5: 24, 6: 120}[n]        # (n-1)!


def test_comc_bad_arguments(bg):
    with pytest.raises(bg.BgError):
        bg.bg_comc_program_stats(9, 4, np.array([9, 0, 0, 0, 0, 0, 0, 0, 0]))
    with pytest.raises(bg.BgError):
        bg.bg_comc_program_stats(6, 4, np.array([5, 0, 0, 0, 0, 0, 0, 0, 0]))
