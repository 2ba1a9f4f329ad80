"""Host-side checks of the seeded input generators (no method arithmetic): RAMBO kinematics, cuts, helicity and
colour rejection rules (readings g8, g9), prefix/chunk reproducibility, SoA packing."""
import itertools

import numpy as np
import pytest


def test_rambo_kinematics_and_cuts(wl):
    for n in (4, 6, 9, 12):
        mom = wl.rambo(n, 20000 if n == 4 else 2000, seed=1, stream=n)
        assert mom.shape[1:] == (n, 4)
        m2 = mom[..., 0] ** 2 - (mom[..., 1:] ** 2).sum(-1)
        assert np.max(np.abs(m2)) < 1e-13 * wl.SQRT_S ** 2                # massless
        assert np.max(np.abs(mom.sum(1))) < 1e-13 * wl.SQRT_S             # momentum conservation, all-outgoing
        assert np.all(mom[:, :2, 0] < 0) and np.all(mom[:, 2:, 0] > 0)
        out = mom[:, 2:]
        pt = np.hypot(out[..., 1], out[..., 2])
        assert pt.min() > wl.PT_MIN
        y = 0.5 * np.log((out[..., 0] + out[..., 3]) / (out[..., 0] - out[..., 3]))
        phi = np.arctan2(out[..., 2], out[..., 1])
        for i, j in itertools.combinations(range(n - 2), 2):
            dphi = np.abs(phi[:, i] - phi[:, j])
            dphi = np.where(dphi > np.pi, 2 * np.pi - dphi, dphi)
            assert np.min(np.hypot(y[:, i] - y[:, j], dphi)) > wl.DR_MIN


def test_prefix_and_chunk_reproducibility(wl):
    a = wl.config_events(1, N=300)
    b = wl.config_events(1, N=100)
    c = wl.config_events(1, N=50, first_event=100)
    assert np.array_equal(a.mom[:100], b.mom) and np.array_equal(a.hel[:100], b.hel)
    assert np.array_equal(a.col[:100], b.col)
    assert np.array_equal(a.mom[100:150], c.mom) and np.array_equal(a.col[100:150], c.col)
    d = wl.config_events(1, N=100, seed=2)
    assert not np.array_equal(d.mom, b.mom)


def test_helicity_rule(wl):
    h = wl.helicities(6, 5000)
    assert set(np.unique(h)) == {-1, 1}
    plus = (h > 0).sum(1)
    assert plus.min() >= 2 and plus.max() <= 4
    raw = wl.helicities(6, 5000, reject_zero=False)
    frac_zero = np.mean(((raw > 0).sum(1) < 2) | ((raw < 0).sum(1) < 2))
    assert abs(frac_zero - 14 / 64) < 0.03                 # (2 + 2n)/2^n at n = 6


def test_colour_rule_sampled(wl):
    col, trials = wl.colours(6, 4000, return_trials=True)
    assert col.min() >= 1 and col.max() <= 3
    for c in col[:200]:
        assert sorted(c[:, 0]) == sorted(c[:, 1])
        assert wl.colour_valid(c)
    assert 0.03 < 1.0 / trials.mean() < 0.08               # acceptance about 5 % of uniform draws


def test_colour_rule_is_exactly_the_nonzero_set_n4(wl, oracle):
    """Reading g8 pinned: an assignment passes the rule iff the colour-dressed amplitude is not identically zero."""
    n = 4
    cols = np.array(list(itertools.product(range(1, 4), repeat=2 * n)), dtype=np.int8).reshape(-1, n, 2)
    valid = np.array([wl.colour_valid(c) for c in cols])
    mom = wl.rambo(n, 1, seed=8, stream=99, ptmin=0, drmin=0)[0]
    N = cols.shape[0]
    tot = np.zeros(N)
    for h in ((1, 1, -1, -1), (1, -1, 1, -1), (1, -1, -1, 1)):
        tot += oracle.cdbg(np.broadcast_to(mom, (N, n, 4)).copy(),
                           np.broadcast_to(np.array(h, dtype=np.int8), (N, n)).copy(), cols)
    assert valid.sum() == 378                               # survey-time count for n = 4
    assert np.all(tot[~valid] < 1e-25 * tot.max())
    assert np.all(tot[valid] > 1e-12 * tot.max())


def test_to_soa(wl):
    ev = wl.config_events(1, N=7)
    mom, hel, col = wl.to_soa(ev.mom, ev.hel, ev.col)
    assert mom.shape == (6, 4, 7) and hel.shape == (6, 7) and col.shape == (6, 2, 7)
    assert mom[3, 2, 5] == ev.mom[5, 3, 2] and hel[4, 6] == ev.hel[6, 4] and col[2, 1, 3] == ev.col[3, 2, 1]
    assert mom.flags.c_contiguous
