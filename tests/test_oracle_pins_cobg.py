"""Pins for the oracle's colour-ordered recursion (Eq. 20-26 of PAPER.md) against what mathematics fixes:
Parke-Taylor moduli (ref. [59]), vanishing helicity configurations, cyclic / reflection / U(1)
identities, gauge invariance, V4 form == tensor form, transversality of the polarisation vectors.
None of these retype the oracle's formulas: each would fail on a dropped term, wrong sign or swapped index."""
import itertools

import numpy as np
import pytest


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def sij(mom, i, j):
    q = mom[i] + mom[j]
    return mdot(q, q)


def parke_taylor_sq(mom, order, i, j):
    """|A(..i-..j-..)|^2 = s_ij^4 / prod_k s_{k,k+1} over the cyclic order (unit normalisation, g_s = 1)."""
    n = len(order)
    den = 1.0
    for k in range(n):
        den *= sij(mom, order[k], order[(k + 1) % n])
    return sij(mom, i, j) ** 4 / den


@pytest.fixture(scope="module")
def events(wl):
    return {n: wl.rambo(n, 6, seed=11, stream=7000 + n) for n in range(4, 9)}


def test_polarisation_vectors(oracle, events):
    for n, moms in events.items():
        for p in moms[0]:
            ep, em = oracle.polarisation(p, +1), oracle.polarisation(p, -1)
            scale = abs(p[0])
            assert abs(mdot(ep, p)) < 1e-13 * scale and abs(mdot(em, p)) < 1e-13 * scale   # transverse
            assert abs(mdot(ep, ep)) < 1e-14 and abs(mdot(em, em)) < 1e-14                    # null
            assert abs(mdot(ep, np.conj(ep)) + 1) < 1e-14                                     # normalised
            assert np.allclose(em, -np.conj(ep), atol=1e-16)      # eps^- = -(eps^+)^* in this phase convention
            assert ep[0] == 0
            # dyadic sum = light-cone projector with k = (q0, -q), Eq. 2-3
            q = p if p[0] > 0 else -p
            k = np.array([q[0], -q[1], -q[2], -q[3]])
            g = np.diag([1.0, -1, -1, -1])
            proj = -g + (np.outer(q, k) + np.outer(k, q)) / mdot(q, k)
            dy = np.outer(ep, np.conj(ep)) + np.outer(em, np.conj(em))
            assert np.allclose(dy, proj, atol=1e-13)


@pytest.mark.parametrize("n", [4, 5, 6, 7, 8])
def test_parke_taylor_all_mhv(oracle, events, n):
    mom = events[n][1]
    order = np.arange(n)
    for i, j in itertools.combinations(range(n), 2):
        for sign in (+1, -1):            # MHV and, by parity, anti-MHV
            hel = np.full(n, sign, dtype=np.int8)
            hel[i] = hel[j] = -sign
            a = oracle.cobg_amp(mom, hel, order)
            assert abs(a) ** 2 == pytest.approx(parke_taylor_sq(mom, order, i, j), rel=2e-11)


def test_parke_taylor_permuted_order(oracle, events):
    mom = events[6][2]
    rng = np.random.default_rng(5)
    for _ in range(5):
        order = rng.permutation(6).astype(np.int32)
        hel = np.array([1, -1, 1, 1, -1, 1], dtype=np.int8)
        a = oracle.cobg_amp(mom, hel, order)
        assert abs(a) ** 2 == pytest.approx(parke_taylor_sq(mom, order, 1, 4), rel=2e-11)


@pytest.mark.parametrize("n", [4, 5, 6, 7])
def test_vanishing_helicity_configurations(oracle, events, n):
    mom = events[n][0]
    order = np.arange(n)
    hel = np.ones(n, dtype=np.int8)
    hel[0] = hel[1] = -1
    typical = abs(oracle.cobg_amp(mom, hel, order))
    for sign in (+1, -1):
        hel = np.full(n, sign, dtype=np.int8)
        assert abs(oracle.cobg_amp(mom, hel, order)) < 1e-11 * typical
        for k in range(n):
            h = hel.copy()
            h[k] = -sign
            assert abs(oracle.cobg_amp(mom, h, order)) < 1e-11 * typical


@pytest.mark.parametrize("n", [5, 6, 7])
def test_cyclic_reflection_u1(oracle, events, n):
    mom = events[n][3]
    rng = np.random.default_rng(n)
    hel = np.array([1, -1, -1, 1, -1, 1, 1][:n], dtype=np.int8)
    order = np.arange(n)
    a = oracle.cobg_amp(mom, hel, order)
    # cyclicity A(1..n) = A(2..n,1)
    assert oracle.cobg_amp(mom, hel, np.roll(order, -1)) == pytest.approx(a, rel=1e-10)
    assert oracle.cobg_amp(mom, hel, np.roll(order, -3)) == pytest.approx(a, rel=1e-10)
    # reflection A(1..n) = (-1)^n A(n..1)
    assert oracle.cobg_amp(mom, hel, order[::-1].copy()) == pytest.approx((-1) ** n * a, rel=1e-10)
    # U(1) decoupling: gluon 0 inserted in every slot of the cyclic order of the others sums to zero
    others = list(range(1, n))
    tot = 0
    for pos in range(n - 1):
        o = others[:pos] + [0] + others[pos:]
        tot += oracle.cobg_amp(mom, hel, np.array(o, dtype=np.int32))
    assert abs(tot) < 1e-10 * abs(a)


@pytest.mark.parametrize("n", [4, 5, 6, 7])
def test_gauge_invariance(oracle, events, n):
    mom = events[n][4]
    hel = np.array([-1, 1, -1, 1, 1, -1, 1][:n], dtype=np.int8)
    ext = np.array([oracle.polarisation(mom[k], hel[k]) for k in range(n)])
    a = oracle.cobg_amp_ext(mom, ext)
    assert a == pytest.approx(oracle.cobg_amp(mom, hel, np.arange(n)), rel=1e-13)
    for k in (0, 2, n - 1):
        e2 = ext.copy()
        e2[k] = mom[k] / abs(mom[k][0])           # eps_k -> p_k: Ward identity
        assert abs(oracle.cobg_amp_ext(mom, e2)) < 1e-11 * abs(a)
        e3 = ext.copy()
        e3[k] = ext[k] + (0.37 - 0.21j) * mom[k] / abs(mom[k][0])   # change of gauge vector
        assert oracle.cobg_amp_ext(mom, e3) == pytest.approx(a, rel=1e-10)


@pytest.mark.parametrize("n", [4, 5, 7, 9])
def test_v4_form_equals_tensor_form(oracle, wl, n):
    mom = wl.rambo(n, 2, seed=3, stream=7100 + n)[1]
    hel = np.array([1, -1, -1, 1, -1, 1, 1, -1, 1][:n], dtype=np.int8)
    order = np.arange(n)
    a = oracle.cobg_amp(mom, hel, order, tensor_form=False)
    b = oracle.cobg_amp(mom, hel, order, tensor_form=True)
    assert b == pytest.approx(a, rel=1e-11)
    # and the extended-precision build of the same source agrees with the double build
    c = oracle.cobg_amp(mom, hel, order, prec="long double")
    assert c == pytest.approx(a, rel=1e-11)


def test_scaling_dimension(oracle, events):
    # A_n has mass dimension 4-n
    mom = events[6][5]
    hel = np.array([1, -1, -1, 1, -1, 1], dtype=np.int8)
    a = oracle.cobg_amp(mom, hel, np.arange(6))
    b = oracle.cobg_amp(2.5 * mom, hel, np.arange(6))
    assert abs(b) == pytest.approx(abs(a) * 2.5 ** (4 - 6), rel=1e-12)
