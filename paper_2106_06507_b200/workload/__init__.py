"""Seeded synthetic workloads (inputs only) shared by the oracle tests, the GPU tests and bench.py.

This module holds none of the method's arithmetic: it draws phase-space points (RAMBO, the paper's event
source), applies the cuts (PAPER.md:L331-334 with BASELINE.json's values) and draws discrete
helicities and colour-flow indices.  The numbers come from ``gen.c`` (built here with gcc on first use).

Arrays are returned in AoS order ``mom[N][n][4]``, ``hel[N][n]``, ``col[N][n][2]``; :func:`to_soa` gives the
event-fastest storage the C-ABI of the CUDA library takes (``include/bg.h``).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libbgworkload.so")
_SRC_PATH = os.path.join(_HERE, "gen.c")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(_SRC_PATH):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", _SRC_PATH, "-o", _LIB_PATH, "-lm"]
        )
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        u64, i32, i64, dbl = ctypes.c_uint64, ctypes.c_int, ctypes.c_longlong, ctypes.c_double
        vp = ctypes.c_void_p
        lib.wl_rambo.argtypes = [u64, u64, i32, i64, i64, dbl, dbl, dbl, vp, vp]
        lib.wl_helicities.argtypes = [u64, u64, i32, i64, i64, i32, vp]
        lib.wl_colours.argtypes = [u64, u64, i32, i64, i64, vp, vp]
        lib.wl_colour_valid.argtypes = [i32, vp]
        for f in (lib.wl_rambo, lib.wl_helicities, lib.wl_colours, lib.wl_colour_valid):
            f.restype = i32
        _lib = lib
    return _lib


SQRT_S = 1000.0  # GeV, BASELINE.json
PT_MIN = 20.0
DR_MIN = 0.4


def rambo(n: int, N: int, seed: int = 1, stream: int = 0, first_event: int = 0, sqrt_s: float = SQRT_S,
          ptmin: float = PT_MIN, drmin: float = DR_MIN, return_trials: bool = False):
    lib = _load()
    mom = np.empty((N, n, 4), dtype=np.float64)
    trials = np.empty(N, dtype=np.int32)
    rc = lib.wl_rambo(seed, stream, n, N, first_event, sqrt_s, ptmin, drmin, mom.ctypes.data, trials.ctypes.data)
    if rc != 0:
        raise ValueError("wl_rambo: bad arguments")
    return (mom, trials) if return_trials else mom


def helicities(n: int, N: int, seed: int = 1, stream: int = 0, first_event: int = 0, reject_zero: bool = True):
    lib = _load()
    hel = np.empty((N, n), dtype=np.int8)
    rc = lib.wl_helicities(seed, stream + (1 << 20), n, N, first_event, int(reject_zero), hel.ctypes.data)
    if rc != 0:
        raise ValueError("wl_helicities: bad arguments")
    return hel


def colours(n: int, N: int, seed: int = 1, stream: int = 0, first_event: int = 0, return_trials: bool = False):
    lib = _load()
    col = np.empty((N, n, 2), dtype=np.int8)
    trials = np.empty(N, dtype=np.int32)
    rc = lib.wl_colours(seed, stream + (2 << 20), n, N, first_event, col.ctypes.data, trials.ctypes.data)
    if rc != 0:
        raise ValueError("wl_colours: bad arguments")
    return (col, trials) if return_trials else col


def colour_valid(col_one_event: np.ndarray) -> bool:
    lib = _load()
    c = np.ascontiguousarray(col_one_event, dtype=np.int8)
    rc = lib.wl_colour_valid(c.shape[0], c.ctypes.data)
    if rc < 0:
        raise ValueError("wl_colour_valid: bad arguments")
    return bool(rc)


def continuous_states(n: int, N: int, seed: int = 1, stream: int = 0):
    """Continuous sampling variables of the paper's CD_MC (Eq. 7, 9, 12; L60-107): one polarisation angle
    phi in [0, 2 pi) per gluon and two unit 3-vectors (eta, etabar), uniform on the sphere, per gluon.
    Returns phi[N][n], eta[N][n][2][3].  Inputs only (seeded numpy generator, independent of the phase-space draw)."""
    rng = np.random.default_rng([seed, stream, n, 0xC0])
    phi = rng.uniform(0.0, 2.0 * np.pi, size=(N, n))
    eta = rng.normal(size=(N, n, 2, 3))
    eta /= np.linalg.norm(eta, axis=-1, keepdims=True)
    return phi, eta


def continuous_to_soa(phi, eta):
    """phi[N][n] -> [n][N]; eta[N][n][2][3] -> [n][6][N] (eta then etabar), as bg_eval_continuous takes them."""
    N, n = phi.shape
    return (np.ascontiguousarray(phi.T), np.ascontiguousarray(np.transpose(eta.reshape(N, n, 6), (1, 2, 0))))


def to_soa(mom=None, hel=None, col=None):
    """AoS [N][n][...] -> event-fastest storage [n][...][N] (C-contiguous), as include/bg.h specifies."""
    out = []
    if mom is not None:
        out.append(np.ascontiguousarray(np.transpose(mom, (1, 2, 0))))
    if hel is not None:
        out.append(np.ascontiguousarray(np.transpose(hel, (1, 0))))
    if col is not None:
        out.append(np.ascontiguousarray(np.transpose(col, (1, 2, 0))))
    return out[0] if len(out) == 1 else tuple(out)


@dataclass
class Events:
    n: int
    mom: np.ndarray            # [N][n][4] float64
    hel: np.ndarray | None     # [N][n] int8 or None (helicity-summed)
    col: np.ndarray | None     # [N][n][2] int8 or None (colour-summed)
    name: str = ""

    @property
    def N(self) -> int:
        return self.mom.shape[0]

    def head(self, k: int) -> "Events":
        return Events(self.n, self.mom[:k], None if self.hel is None else self.hel[:k],
                      None if self.col is None else self.col[:k], self.name)

    def take(self, idx) -> "Events":
        return Events(self.n, self.mom[idx], None if self.hel is None else self.hel[idx],
                      None if self.col is None else self.col[idx], self.name)


# BASELINE.json configs (index = position in BASELINE.json "configs").
def config_events(config: int, N: int | None = None, n: int | None = None, seed: int = 1,
                  first_event: int = 0) -> Events:
    """The five BASELINE.json workloads.  ``N`` overrides the event count (prefix property: the first k events
    of a larger draw equal a draw of k events)."""
    if config == 0:      # n=4 COBG, helicity- and colour-summed, no cuts
        N = 1024 if N is None else N
        return Events(4, rambo(4, N, seed, 100, first_event, ptmin=0.0, drmin=0.0), None, None, "C1 n=4 COBG helsum")
    if config == 1:      # n=6 CDBG sampled
        N = (1 << 20) if N is None else N
        return Events(6, rambo(6, N, seed, 200, first_event), helicities(6, N, seed, 200, first_event),
                      colours(6, N, seed, 200, first_event), "C2 n=6 CDBG sampled")
    if config == 2:      # n=7 COBG, sampled helicities, full colour
        N = (1 << 18) if N is None else N
        return Events(7, rambo(7, N, seed, 300, first_event), helicities(7, N, seed, 300, first_event), None,
                      "C3 n=7 COBG full colour")
    if config == 3:      # n=9 CDBG sampled
        N = (1 << 18) if N is None else N
        return Events(9, rambo(9, N, seed, 400, first_event), helicities(9, N, seed, 400, first_event),
                      colours(9, N, seed, 400, first_event), "C4 n=9 CDBG sampled")
    if config == 4:      # n=4..12 sweep, CDBG sampled
        if n is None:
            raise ValueError("config 4 (sweep) needs n")
        N = (1 << 16) if N is None else N
        s = 500 + n
        return Events(n, rambo(n, N, seed, s, first_event), helicities(n, N, seed, s, first_event),
                      colours(n, N, seed, s, first_event), f"C5 n={n} CDBG sampled")
    raise ValueError("config must be 0..4")
