"""Pins of the oracle's colour-dressed recursion with general external states (continuous colour and polarisation
sampling, Eq. 5-14).  Nothing here touches the CUDA path."""
import itertools

import numpy as np
import pytest


def random_states(rng, N, n):
    phi = rng.uniform(0, 2 * np.pi, size=(N, n))
    eta = rng.normal(size=(N, n, 2, 3))
    eta /= np.linalg.norm(eta, axis=-1, keepdims=True)      # two unit 3-vectors per gluon (Eq. 9)
    return phi, eta


def elementary(i, j):
    X = np.zeros((3, 3), dtype=complex)
    X[i, j] = 1.0
    return X


@pytest.mark.parametrize("n", [4, 5, 6, 7])
def test_elementary_colour_matrices_reproduce_the_discrete_recursion(oracle, wl, n):
    """X_k = e_{i_k j_k} and eps^lambda as external states is the pinned discrete CDBG."""
    ev = wl.config_events(4, N=40, n=n)
    ext = np.array([[oracle.polarisation(ev.mom[e, k], int(ev.hel[e, k])) for k in range(n)] for e in range(ev.N)])
    X = np.array([[elementary(ev.col[e, k, 0] - 1, ev.col[e, k, 1] - 1) for k in range(n)] for e in range(ev.N)])
    got = np.abs(oracle.cdbg_general(ev.mom, ext, X)) ** 2
    ref = oracle.cdbg(ev.mom, ev.hel, ev.col)
    assert np.allclose(got, ref, rtol=1e-12, atol=0)


def test_multilinear_in_the_colour_matrices_n4(oracle, wl):
    """Eq. 14: A(X_1..X_n) = sum over all 9^n elementary assignments of prod_k X_k[i_k][j_k] A_{i1 j1 .. in jn}."""
    rng = np.random.default_rng(11)
    ev = wl.config_events(4, N=1, n=4)
    mom = ev.mom[0]
    ext = np.array([oracle.polarisation(mom[k], int(ev.hel[0, k])) for k in range(4)])
    X = rng.normal(size=(4, 3, 3)) + 1j * rng.normal(size=(4, 3, 3))
    full = oracle.cdbg_general(mom[None], ext[None], X[None])[0]
    pairs = list(itertools.product(range(3), repeat=2))
    combos = list(itertools.product(pairs, repeat=4))
    Xs = np.array([[elementary(*c[k]) for k in range(4)] for c in combos])
    amps = oracle.cdbg_general(np.broadcast_to(mom, (len(combos), 4, 4)).copy(),
                               np.broadcast_to(ext, (len(combos), 4, 4)).copy(), Xs)
    coef = np.array([np.prod([X[k][c[k]] for k in range(4)]) for c in combos])
    assert abs(np.sum(coef * amps) - full) <= 1e-11 * abs(full)


@pytest.mark.parametrize("n", [4, 5, 6])
def test_real_polarisation_is_the_helicity_superposition(oracle, wl, n):
    """e(phi) = cos(phi) e1 + sin(phi) e2 = (e^{i phi} eps^- - e^{-i phi} eps^+)/sqrt2 (Eq. 5, 7 with the unit
    vectors of reading g2): the amplitude is the corresponding superposition of the 2^n helicity amplitudes."""
    rng = np.random.default_rng(5)
    ev = wl.config_events(4, N=1, n=n)
    mom = ev.mom[0]
    phi, eta = random_states(rng, 1, n)
    ext, X = oracle.continuous_states(mom[None], phi, eta)
    full = oracle.cdbg_general(mom[None], ext, X)[0]
    tot = 0.0
    for lam in itertools.product((-1, 1), repeat=n):
        e = np.array([oracle.polarisation(mom[k], lam[k]) for k in range(n)])
        c = np.prod([(np.exp(1j * phi[0, k]) if lam[k] < 0 else -np.exp(-1j * phi[0, k])) / np.sqrt(2.0)
                     for k in range(n)])
        tot += c * oracle.cdbg_general(mom[None], e[None], X)[0]
    assert abs(tot - full) <= 1e-11 * abs(full)


@pytest.mark.parametrize("n", [4, 6, 8])
def test_real_states_give_real_amplitudes_and_the_trace_part_decouples(oracle, wl, n):
    """PAPER.md:L66 "real valued amplitudes for the gluon-only case"; the U(1) part of
    eta_i T^a_ij etabar_j T^a_hg = eta_g etabar_h - delta_hg (eta.etabar)/3 does not couple to gluons."""
    rng = np.random.default_rng(n)
    ev = wl.config_events(4, N=6, n=n)
    phi, eta = random_states(rng, ev.N, n)
    ext, X = oracle.continuous_states(ev.mom, phi, eta)
    A = oracle.cdbg_general(ev.mom, ext, X)
    assert np.all(np.abs(A.imag) <= 1e-12 * np.abs(A.real))
    dots = np.einsum("ekc,ekc->ek", eta[:, :, 0, :], eta[:, :, 1, :])
    Xt = X - dots[:, :, None, None] * np.eye(3)[None, None] / 3.0
    At = oracle.cdbg_general(ev.mom, ext, Xt)
    assert np.all(np.abs(At - A) <= 1e-10 * np.abs(A))
    assert np.allclose(oracle.cdbg_continuous(ev.mom, phi, eta), np.abs(A) ** 2, rtol=1e-14)


def test_monte_carlo_normalisation_of_eq13_n4(oracle):
    """Eq. 8-13: averaging |A|^2 over phi (uniform) and the two unit vectors per gluon (uniform on the sphere), times
    (2 x 3 x 3)^n, estimates the helicity- and colour-summed |M|^2: 7776 at the exact gg -> gg point of the golden file.
    Statistical pin of the normalisation (a wrong factor per gluon would be off by 2^4 or more)."""
    rng = np.random.default_rng(2024)
    mom = np.array([[-4, 0, 0, -4], [-2, 0, 0, 2], [3, 2, 2, 1], [3, -2, -2, 1]], dtype=float)
    N = 400000
    phi, eta = random_states(rng, N, 4)
    # continuous_states loops in Python: build the states vectorised here from the same definitions
    ep = np.array([oracle.polarisation(mom[k], +1) for k in range(4)])
    em = np.array([oracle.polarisation(mom[k], -1) for k in range(4)])
    e1, e2 = (em - ep) / np.sqrt(2.0), 1j * (ep + em) / np.sqrt(2.0)
    ext = np.cos(phi)[:, :, None] * e1[None] + np.sin(phi)[:, :, None] * e2[None]
    X = np.einsum("ekh,ekg->ekhg", eta[:, :, 1, :], eta[:, :, 0, :]).astype(complex)
    w = np.abs(oracle.cdbg_general(np.broadcast_to(mom, (N, 4, 4)).copy(), ext, X)) ** 2 * 18.0 ** 4
    est, err = w.mean(), w.std() / np.sqrt(N)
    assert abs(est - 7776.0) < 5 * err and err < 0.05 * 7776.0
