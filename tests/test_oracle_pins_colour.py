"""Pins for the oracle's colour treatment: colour matrix Eq. 17, full-colour sum Eq. 16 against the closed-form
gg->gg result (refs. [52,53]; BASELINE.json north_star), leading-colour formula Eq. 33, and the
colour-dressed recursion Eq. 28-32 against its definition Eq. 19 and against the explicit colour sum."""
import itertools
import math
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def gg_gg_closed_form(mom):
    """Helicity- and colour-summed |M|^2 at g_s = 1, no averaging: 256 x (9/2)(3 - tu/s^2 - su/t^2 - st/u^2)."""
    s = mdot(mom[0] + mom[1], mom[0] + mom[1])
    t = mdot(mom[0] + mom[2], mom[0] + mom[2])
    u = mdot(mom[0] + mom[3], mom[0] + mom[3])
    return 1152.0 * (3 - t * u / s ** 2 - s * u / t ** 2 - s * t / u ** 2)


def test_colour_matrix_n4_n5_hand_values(oracle):
    # C_A = 2 N_c = 6 in the Tr(T^a T^b) = delta^ab normalisation: diag = C_A^2 (N_c^2-1), off-diag = half of it
    assert np.array_equal(oracle.colour_matrix(4), np.array([[288.0, 144.0], [144.0, 288.0]]))
    ref5 = 432 * np.array([[4, 2, 2, 1, 1, 0], [2, 4, 1, 0, 2, 1], [2, 1, 4, 2, 0, 1],
                           [1, 0, 2, 4, 1, 2], [1, 2, 0, 1, 4, 2], [0, 1, 1, 2, 2, 4]], dtype=float)
    assert np.array_equal(oracle.colour_matrix(5), ref5)


@pytest.mark.parametrize("n", [4, 5, 6, 7])
def test_colour_matrix_structure(oracle, n):
    C = oracle.colour_matrix(n)
    m = math.factorial(n - 2)
    assert C.shape == (m, m)
    assert np.array_equal(C, C.T)
    assert np.all(np.diag(C) == 6 ** (n - 2) * 8)            # C_A^{n-2} (N_c^2 - 1)
    # C_{sigma sigma'} depends only on sigma^-1 sigma' (relabelling invariance, PAPER.md:L321 footnote 3)
    perms = list(itertools.permutations(range(n - 2)))
    index = {p: i for i, p in enumerate(perms)}
    for a in range(0, m, max(1, m // 7)):
        for b in range(0, m, max(1, m // 5)):
            inv = np.argsort(perms[a])
            rel = tuple(int(inv[x]) for x in perms[b])
            assert C[a, b] == C[0, index[rel]]
    # positive definite for n <= 5; positive semi-definite in general (it is a Gram matrix)
    ev = np.linalg.eigvalsh(C)
    assert ev.min() > -1e-6 * ev.max()


def test_gg_gg_closed_form_golden(oracle):
    # exactly representable momenta: s = 32, t = u = -16 -> 1152 * 6.75 = 7776 exactly
    rows = [l.split() for l in open(os.path.join(GOLDEN, "gg_gg_exact.txt")) if l.strip() and not l.startswith("#")]
    mom = np.array([[float(x) for x in r] for r in rows[:4]])
    expect = float(rows[4][0])
    assert gg_gg_closed_form(mom) == expect
    got = oracle.cobg_full_colour(mom[None])[0]
    assert got == pytest.approx(expect, rel=1e-13)
    assert oracle.cobg_full_colour(mom[None], tensor_form=True)[0] == pytest.approx(expect, rel=1e-13)


def test_gg_gg_closed_form_rambo(oracle, wl):
    ev = wl.config_events(0, N=64)
    got = oracle.cobg_full_colour(ev.mom)
    ref = np.array([gg_gg_closed_form(m) for m in ev.mom])
    assert np.max(np.abs(got / ref - 1)) < 1e-11
    got_ld = oracle.cobg_full_colour(ev.mom, prec="long double")
    assert np.max(np.abs(got_ld / ref - 1)) < 1e-11


@pytest.mark.parametrize("n", [4, 5])
def test_leading_colour_formula_exact_at_n4_n5(oracle, wl, n):
    """Eq. 33 without its O(1/N^2) remainder equals the full-colour sum exactly for n = 4, 5."""
    mom = wl.rambo(n, 1, seed=2, stream=7200 + n)[0]
    hel = np.array([1, -1, -1, 1, 1][:n], dtype=np.int8)
    full = oracle.cobg_full_colour(mom[None], hel[None])[0]
    lc = 0.0
    for sig in itertools.permutations(range(1, n)):
        lc += abs(oracle.cobg_amp(mom, hel, np.array((0,) + sig, dtype=np.int32))) ** 2
    lc *= 3 ** (n - 2) * 8
    assert lc == pytest.approx(full, rel=1e-11)


def test_leading_colour_not_exact_at_n6(oracle, wl):
    mom = wl.rambo(6, 1, seed=2, stream=7206)[0]
    hel = np.array([1, -1, -1, 1, 1, -1], dtype=np.int8)
    full = oracle.cobg_full_colour(mom[None], hel[None])[0]
    lc = sum(abs(oracle.cobg_amp(mom, hel, np.array((0,) + s, dtype=np.int32))) ** 2
             for s in itertools.permutations(range(1, 6))) * 3 ** 4 * 8
    assert 0.5 < lc / full < 1.5 and abs(lc / full - 1) > 1e-3


@pytest.mark.parametrize("n", [4, 5])
def test_sum_over_all_colour_flows_equals_full_colour(oracle, wl, n):
    """Eq. 11: summing |A_{i1j1..injn}|^2 over all 9^n colour-flow assignments gives the adjoint colour sum."""
    mom = wl.rambo(n, 1, seed=4, stream=7300 + n)[0]
    hel = np.array([1, -1, 1, -1, -1][:n], dtype=np.int8)
    cols = np.array(list(itertools.product(range(1, 4), repeat=2 * n)), dtype=np.int8).reshape(-1, n, 2)
    N = cols.shape[0]
    moms = np.broadcast_to(mom, (N, n, 4)).copy()
    hels = np.broadcast_to(hel, (N, n)).copy()
    tot = oracle.cdbg(moms, hels, cols).sum()
    full = oracle.cobg_full_colour(mom[None], hel[None])[0]
    assert tot == pytest.approx(full, rel=1e-11)


def test_n4_full_sum_via_colour_dressed_equals_closed_form(oracle, wl):
    mom = wl.config_events(0, N=3).mom[2]
    cols = np.array(list(itertools.product(range(1, 4), repeat=8)), dtype=np.int8).reshape(-1, 4, 2)
    N = cols.shape[0]
    moms = np.broadcast_to(mom, (N, 4, 4)).copy()
    tot = 0.0
    for h in itertools.product((-1, 1), repeat=4):
        tot += oracle.cdbg(moms, np.broadcast_to(np.array(h, dtype=np.int8), (N, 4)).copy(), cols).sum()
    assert tot == pytest.approx(gg_gg_closed_form(mom), rel=1e-11)


@pytest.mark.parametrize("n", [4, 5, 6, 7, 8])
def test_colour_dressed_equals_colour_flow_definition(oracle, wl, n):
    ev = wl.config_events(4, N=48, n=n, seed=9)
    a = oracle.cdbg(ev.mom, ev.hel, ev.col)
    b, cnt = oracle.colour_flow(ev.mom, ev.hel, ev.col, return_count=True)
    assert np.all(cnt >= 1)
    # truth in extended precision; compare well-conditioned events tightly, the rest through the truth
    t = oracle.colour_flow(ev.mom, ev.hel, ev.col, prec="long double")
    ta = oracle.cdbg(ev.mom, ev.hel, ev.col, prec="long double")
    assert np.max(np.abs(ta - t) / t) < 1e-13          # the two formulations agree in extended precision
    assert np.max(np.abs(a - t) / t) < 1e-9 and np.median(np.abs(a - t) / t) < 1e-13
    assert np.max(np.abs(b - t) / t) < 1e-9


def test_colour_dressed_invariances(oracle, wl):
    n = 6
    ev = wl.config_events(1, N=24, seed=5)
    base = oracle.cdbg(ev.mom, ev.hel, ev.col, prec="long double")
    rng = np.random.default_rng(1)
    # relabel gluons (exercises subset order and the choice of the contracted leg)
    perm = rng.permutation(n)
    assert np.allclose(oracle.cdbg(ev.mom[:, perm], ev.hel[:, perm], ev.col[:, perm], prec="long double"), base,
                       rtol=1e-12)
    # i <-> j on all gluons (charge conjugation), permutation of colour labels, all helicities flipped
    assert np.allclose(oracle.cdbg(ev.mom, ev.hel, ev.col[:, :, ::-1].copy(), prec="long double"), base, rtol=1e-12)
    relabel = np.array([0, 3, 1, 2], dtype=np.int8)
    assert np.allclose(oracle.cdbg(ev.mom, ev.hel, relabel[ev.col], prec="long double"), base, rtol=1e-12)
    assert np.allclose(oracle.cdbg(ev.mom, -ev.hel, ev.col, prec="long double"), base, rtol=1e-12)
    # rotation of all momenta, and dimension: |A|^2 -> kappa^{-2(n-4)} |A|^2
    th = 0.7
    R = np.eye(4)
    R[1, 1], R[1, 3], R[3, 1], R[3, 3] = math.cos(th), math.sin(th), -math.sin(th), math.cos(th)
    assert np.allclose(oracle.cdbg(ev.mom @ R.T, ev.hel, ev.col, prec="long double"), base, rtol=1e-10)
    assert np.allclose(oracle.cdbg(3.0 * ev.mom, ev.hel, ev.col, prec="long double"), base * 3.0 ** (-2 * (n - 4)),
                       rtol=1e-12)


def test_invalid_colours_give_exact_zero(oracle, wl):
    ev = wl.config_events(1, N=4)
    col = ev.col.copy()
    col[:, 0, 0] = (col[:, 0, 0] % 3) + 1          # break multiset{i} == multiset{j}
    assert np.all(oracle.cdbg(ev.mom, ev.hel, col) == 0.0)
