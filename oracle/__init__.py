"""ORACLE — TEST INFRASTRUCTURE ONLY (see bg_oracle.cpp header).

ctypes front end to ``libbgoracle.so`` (plain C++ written from PAPER.md).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this.
It imports nothing from ``paper_2106_06507_b200``.

Arrays are AoS: ``mom[N][n][4]`` float64 (E,px,py,pz; all-outgoing), ``hel[N][n]`` int8 (+1/-1),
``col[N][n][2]`` int8 in {1,2,3}.  ``prec``: ``"double"`` or ``"long double"`` (x87 80-bit, the round-off truth).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bg_oracle.cpp")
_LIB = os.path.join(_HERE, "libbgoracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _LIB])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        for name in ("bgo_polarisation", "bgo_cobg_amp_ext", "bgo_cobg_amp", "bgo_colour_matrix",
                     "bgo_cobg_full_colour", "bgo_cdbg", "bgo_colour_flow", "bgo_max_threads", "bgo_cdbg_general"):
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def _prec(prec: str) -> int:
    return {"double": 0, "long double": 1}[prec]


def _p(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i8(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int8)


def max_threads() -> int:
    return int(_load().bgo_max_threads())


def polarisation(p, lam: int) -> np.ndarray:
    """eps^lam(p) as a complex 4-vector (upper index)."""
    p = _f64(p)
    out = np.empty((4, 2))
    _load().bgo_polarisation(_p(p), ctypes.c_int(int(lam)), _p(out))
    return out[:, 0] + 1j * out[:, 1]


def cobg_amp_ext(mom, ext, tensor_form: bool = False, prec: str = "double") -> complex:
    """Colour-ordered amplitude (Eq. 20/22) for explicit external currents ext[n][4] complex; legs in order."""
    mom = _f64(mom)
    n = mom.shape[0]
    e = np.ascontiguousarray(np.stack([np.real(ext), np.imag(ext)], axis=-1), dtype=np.float64)
    out = np.empty(2)
    rc = _load().bgo_cobg_amp_ext(n, _p(mom), _p(e), int(tensor_form), _prec(prec), _p(out))
    assert rc == 0
    return complex(out[0], out[1])


def cobg_amp(mom, hel, order, tensor_form: bool = False, prec: str = "double") -> complex:
    """A(order[0],..,order[n-1]) for one event; order holds 0-based gluon labels."""
    mom = _f64(mom)
    n = mom.shape[0]
    hel = _i8(hel)
    order = np.ascontiguousarray(order, dtype=np.int32)
    assert order.shape[0] == n
    out = np.empty(2)
    rc = _load().bgo_cobg_amp(n, _p(mom), _p(hel), _p(order), int(tensor_form), _prec(prec), _p(out))
    assert rc == 0
    return complex(out[0], out[1])


_cm_cache: dict[int, np.ndarray] = {}


def colour_matrix(n: int) -> np.ndarray:
    """Eq. 17 from its definition; sigma over permutations of gluons 2..n-1 in lexicographic order."""
    if n not in _cm_cache:
        import math
        m = math.factorial(n - 2)
        C = np.empty((m, m))
        rc = _load().bgo_colour_matrix(n, _p(C))
        assert rc == 0
        # Eq. 17 is integer-valued in this normalisation (a signed sum of powers of N_c); the floating-point
        # evaluation from Gell-Mann matrices carries ~1e-12 noise, removed here after checking it is noise.
        Cr = np.rint(C)
        assert np.max(np.abs(C - Cr)) < 1e-7, "colour matrix not integer-valued"
        _cm_cache[n] = Cr
    return _cm_cache[n]


def cobg_full_colour(mom, hel=None, C=None, tensor_form: bool = False, prec: str = "double", threads: int = 0,
                     return_amps: bool = False):
    """Batched sum_{sigma sigma'} C A A^* (Eq. 16).  hel=None sums all 2^n helicity assignments."""
    mom = _f64(mom)
    N, n = mom.shape[0], mom.shape[1]
    hel = _i8(hel)
    if C is None:
        C = colour_matrix(n)
    C = _f64(C)
    out = np.empty(N)
    amps = None
    if return_amps:
        assert hel is not None
        amps = np.empty((N, C.shape[0], 2))
    rc = _load().bgo_cobg_full_colour(n, ctypes.c_longlong(N), _p(mom), _p(hel), _p(C), int(tensor_form),
                                      _prec(prec), int(threads), _p(out), _p(amps))
    assert rc == 0
    if return_amps:
        return out, amps[..., 0] + 1j * amps[..., 1]
    return out


def cdbg(mom, hel, col, prec: str = "double", threads: int = 0, return_live: bool = False,
         return_rho: bool = False):
    """Batched colour-dressed |A|^2 (Eq. 28-32, colour-flow basis, given helicities and colours).

    ``return_rho`` adds the top-level cancellation ratio rho = |A| / sum_terms |eps_n . term| (terms = the
    ordered-split contributions to the last current), the conditioning measure of DESIGN.md's parity protocol."""
    mom = _f64(mom)
    N, n = mom.shape[0], mom.shape[1]
    hel, col = _i8(hel), _i8(col)
    out = np.empty(N)
    live = np.empty(N, dtype=np.int64)
    rho = np.empty(N)
    rc = _load().bgo_cdbg(n, ctypes.c_longlong(N), _p(mom), _p(hel), _p(col), _prec(prec), int(threads), _p(out),
                          _p(live), _p(rho))
    assert rc == 0
    res = (out,) + ((live,) if return_live else ()) + ((rho,) if return_rho else ())
    return res if len(res) > 1 else out


def cdbg_general(mom, ext, X, prec: str = "double", threads: int = 0) -> np.ndarray:
    """Batched colour-dressed amplitude (complex) for general external states: ext[N][n][4] complex polarisation
    vectors, X[N][n][3][3] complex colour matrices (Eq. 14 + Eq. 28-32)."""
    mom = _f64(mom)
    N, n = mom.shape[0], mom.shape[1]
    e = np.ascontiguousarray(np.stack([np.real(ext), np.imag(ext)], axis=-1), dtype=np.float64)
    x = np.ascontiguousarray(np.stack([np.real(X), np.imag(X)], axis=-1), dtype=np.float64)
    assert e.shape == (N, n, 4, 2) and x.shape == (N, n, 3, 3, 2)
    amp = np.empty((N, 2))
    rc = _load().bgo_cdbg_general(n, ctypes.c_longlong(N), _p(mom), _p(e), _p(x), _prec(prec), int(threads), _p(amp))
    assert rc == 0
    return amp[:, 0] + 1j * amp[:, 1]


def continuous_states(mom, phi, eta):
    """External states of the continuous sampling (Eq. 7, 9, 12): real polarisation e = cos(phi) e1 + sin(phi) e2
    with e1 = (eps^- - eps^+)/sqrt2, e2 = i (eps^+ + eps^-)/sqrt2 (the unit vectors of reading g2), and colour matrix
    X_hg = etabar_h eta_g from eta[..., 0, :] = eta, eta[..., 1, :] = etabar.  Returns (ext, X)."""
    mom = _f64(mom)
    N, n = mom.shape[0], mom.shape[1]
    ext = np.empty((N, n, 4), dtype=complex)
    for e in range(N):
        for k in range(n):
            ep, em = polarisation(mom[e, k], +1), polarisation(mom[e, k], -1)
            e1, e2 = (em - ep) / np.sqrt(2.0), 1j * (ep + em) / np.sqrt(2.0)
            ext[e, k] = np.cos(phi[e, k]) * e1 + np.sin(phi[e, k]) * e2
    X = np.einsum("ekh,ekg->ekhg", eta[:, :, 1, :], eta[:, :, 0, :]).astype(complex)
    return ext, X


def cdbg_continuous(mom, phi, eta, prec: str = "double", threads: int = 0) -> np.ndarray:
    """|A|^2 of the continuous colour / polarisation sub-amplitude (Eq. 14)."""
    ext, X = continuous_states(mom, phi, eta)
    return np.abs(cdbg_general(mom, ext, X, prec=prec, threads=threads)) ** 2


def colour_flow(mom, hel, col, prec: str = "double", threads: int = 0, return_count: bool = False,
                return_rho: bool = False):
    """Batched Eq. 19 brute force: |sum over colour-connected orderings of COBG amplitudes|^2.

    ``return_rho`` adds rho19 = |sum_sigma A_sigma| / sum_sigma |A_sigma|, the cancellation between the colour
    orderings of Eq. 19 (1 = none)."""
    mom = _f64(mom)
    N, n = mom.shape[0], mom.shape[1]
    hel, col = _i8(hel), _i8(col)
    out = np.empty(N)
    cnt = np.empty(N, dtype=np.int64)
    rho = np.empty(N)
    rc = _load().bgo_colour_flow(n, ctypes.c_longlong(N), _p(mom), _p(hel), _p(col), _prec(prec), int(threads),
                                 _p(out), _p(cnt), _p(rho))
    assert rc == 0
    res = (out,) + ((cnt,) if return_count else ()) + ((rho,) if return_rho else ())
    return res if len(res) > 1 else out
