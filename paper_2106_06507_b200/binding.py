"""Thin ctypes binding of libbg.so (include/bg.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of ``csrc/``; there is no CPU or PyTorch fallback.  If the
shared library is missing or cannot be loaded, every entry point raises :class:`BgError` loudly.
PyTorch is used by callers for device buffers and streams only; this module accepts either integers (raw
device pointers) or objects with ``data_ptr()`` (torch tensors) / ``ctypes.data`` (numpy arrays, host calls).
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbg.so")

BG_OK, BG_EINVAL, BG_ENOMEM, BG_ECUDA, BG_EUNSUPPORTED, BG_ELIMIT = 0, -1, -2, -3, -4, -5
BG_STATIC_SCRATCH_BYTES = 32 << 20
BG_REC_COBG, BG_REC_CDBG = 0x001, 0x002
BG_HEL_SUM, BG_HEL_GIVEN = 0x010, 0x020
BG_COL_FULL, BG_COL_GIVEN, BG_COL_LC = 0x100, 0x200, 0x400
BG_COBG_HELSUM_FULLCOLOR = BG_REC_COBG | BG_HEL_SUM | BG_COL_FULL
BG_COBG_HELGIVEN_FULLCOLOR = BG_REC_COBG | BG_HEL_GIVEN | BG_COL_FULL
BG_CDBG_GIVEN = BG_REC_CDBG | BG_HEL_GIVEN | BG_COL_GIVEN
BG_CDBG_HELSUM_COLGIVEN = BG_REC_CDBG | BG_HEL_SUM | BG_COL_GIVEN
BG_HEL_CONT, BG_COL_CONT = 0x040, 0x800
BG_CDBG_CONTINUOUS = BG_REC_CDBG | BG_HEL_CONT | BG_COL_CONT
BG_COMC_GIVEN = BG_REC_COBG | BG_HEL_GIVEN | BG_COL_GIVEN
BG_COBG_HELSUM_LC = BG_REC_COBG | BG_HEL_SUM | BG_COL_LC
BG_COBG_HELGIVEN_LC = BG_REC_COBG | BG_HEL_GIVEN | BG_COL_LC
BG_OPT_KERNEL, BG_OPT_SCRATCH_LIMIT, BG_OPT_LANES, BG_OPT_TIMING, BG_OPT_SMEM_LIMIT, BG_OPT_PRECISION = 1, 2, 3, 4, 5, 6
BG_OPT_FLAG_THRESHOLD, BG_OPT_FLAG_CANCELLATION, BG_OPT_FLAG_TWIN, BG_OPT_FRAME = 7, 8, 9, 10

EXPORTS = ("bg_init", "bg_eval", "bg_eval_continuous", "bg_generate", "bg_colour_rule", "bg_eval_host", "bg_reserve", "bg_scratch_bytes", "bg_current_bytes_per_event",
           "bg_set_option", "bg_colour_matrix", "bg_build_colour_matrix", "bg_last_launch_count",
           "bg_last_kernel_name", "bg_last_kernel_ms", "bg_last_refined", "bg_last_twin", "bg_class_program_stats", "bg_comc_program_stats", "bg_destroy", "bg_strerror", "bg_fp64_peak_probe", "bg_colour_form_probe",
           "bg_static_setup", "bg_static_max_events", "bg_eval_static")


class BgError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {bg_strerror(code) if _lib is not None else code} (code {code})")
        self.code = code


_lib = None


def load():
    """Load libbg.so (built by ``paper_2106_06507_b200.build``); raises if it is absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2106_06507_b200.build` "
                               "(there is no fallback path)")
        lib = ctypes.CDLL(LIB_PATH)
        vp, ll, i = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int
        lib.bg_init.argtypes = [ctypes.POINTER(vp), i, i]
        lib.bg_eval.argtypes = [vp, vp, ll, vp, vp, vp, vp]
        lib.bg_eval_host.argtypes = [vp, ll, vp, vp, vp, vp]
        lib.bg_generate.argtypes = [vp, i, ll, ctypes.c_ulonglong, ctypes.c_ulonglong, ll, ctypes.c_double, ctypes.c_double,
                                    ctypes.c_double, i, vp, vp, vp]
        lib.bg_generate.restype = i
        lib.bg_colour_rule.argtypes = [i, vp]
        lib.bg_colour_rule.restype = i
        lib.bg_eval_continuous.argtypes = [vp, vp, ll, vp, vp, vp, vp]
        lib.bg_eval_continuous.restype = i
        lib.bg_reserve.argtypes = [vp, ll]
        lib.bg_scratch_bytes.argtypes = [vp, ll]
        lib.bg_scratch_bytes.restype = ctypes.c_size_t
        lib.bg_current_bytes_per_event.argtypes = [vp]
        lib.bg_current_bytes_per_event.restype = ctypes.c_size_t
        lib.bg_set_option.argtypes = [vp, i, ll]
        lib.bg_colour_matrix.argtypes = [vp, vp]
        lib.bg_build_colour_matrix.argtypes = [i, vp]
        lib.bg_last_launch_count.argtypes = [vp]
        lib.bg_last_kernel_name.argtypes = [vp]
        lib.bg_last_kernel_name.restype = ctypes.c_char_p
        lib.bg_last_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
        lib.bg_last_kernel_ms.restype = i
        lib.bg_last_refined.argtypes = [vp, ctypes.POINTER(ll), ctypes.POINTER(ctypes.c_double)]
        lib.bg_last_refined.restype = i
        lib.bg_last_twin.argtypes = [vp, ctypes.POINTER(ll)]
        lib.bg_last_twin.restype = i
        lib.bg_class_program_stats.argtypes = [i, i, vp, vp]
        lib.bg_class_program_stats.restype = i
        lib.bg_comc_program_stats.argtypes = [i, i, vp, vp]
        lib.bg_comc_program_stats.restype = i
        lib.bg_destroy.argtypes = [vp]
        lib.bg_strerror.argtypes = [i]
        lib.bg_strerror.restype = ctypes.c_char_p
        lib.bg_fp64_peak_probe.argtypes = [i, ctypes.POINTER(ctypes.c_double)]
        dp = ctypes.POINTER(ctypes.c_double)
        lib.bg_colour_form_probe.argtypes = [i, ll, i, dp, dp, dp, vp, vp]
        lib.bg_colour_form_probe.restype = i
        lib.bg_static_setup.argtypes = []
        lib.bg_static_setup.restype = i
        lib.bg_static_max_events.argtypes = [i]
        lib.bg_static_max_events.restype = ll
        lib.bg_eval_static.argtypes = [vp, i, ll, vp, vp, vp, vp]
        lib.bg_eval_static.restype = i
        for name in ("bg_init", "bg_eval", "bg_eval_host", "bg_reserve", "bg_set_option", "bg_colour_matrix",
                     "bg_build_colour_matrix", "bg_last_launch_count", "bg_destroy", "bg_fp64_peak_probe"):
            getattr(lib, name).restype = i
        _lib = lib
    return _lib


def _ptr(x):
    if x is None:
        return None
    if isinstance(x, int):
        return ctypes.c_void_p(x)
    if hasattr(x, "data_ptr"):
        return ctypes.c_void_p(x.data_ptr())
    if hasattr(x, "ctypes"):
        return ctypes.c_void_p(x.ctypes.data)
    raise TypeError(f"cannot take a pointer from {type(x)}")


def _check(rc: int, what: str):
    if rc != BG_OK:
        raise BgError(rc, what)


def bg_strerror(code: int) -> str:
    return load().bg_strerror(code).decode()


def bg_init(n: int, mode: int):
    ctx = ctypes.c_void_p()
    _check(load().bg_init(ctypes.byref(ctx), n, mode), "bg_init")
    return ctx


def bg_eval(ctx, stream, N: int, mom, hel, col, out) -> None:
    """Device pointers (or torch CUDA tensors); ``stream`` is a cudaStream_t as int (0/None = default stream)."""
    s = ctypes.c_void_p(int(stream)) if stream else None
    _check(load().bg_eval(ctx, s, N, _ptr(mom), _ptr(hel), _ptr(col), _ptr(out)), "bg_eval")


def bg_eval_continuous(ctx, stream, N: int, mom, phi, eta, out) -> None:
    """Device pointers; phi[n][N], eta[n][6][N] (eta then etabar), event-fastest."""
    s = ctypes.c_void_p(int(stream)) if stream else None
    _check(load().bg_eval_continuous(ctx, s, N, _ptr(mom), _ptr(phi), _ptr(eta), _ptr(out)), "bg_eval_continuous")


def bg_generate(stream, n: int, N: int, seed: int, stream_id: int, first_event: int, sqrt_s: float, ptmin: float,
                drmin: float, reject_zero_helicities: bool, mom, hel, col) -> None:
    """Generate N synthetic events on the device into event-fastest buffers (any of mom / hel / col may be None)."""
    s = ctypes.c_void_p(int(stream)) if stream else None
    _check(load().bg_generate(s, n, N, seed, stream_id, first_event, sqrt_s, ptmin, drmin, int(reject_zero_helicities),
                              _ptr(mom), _ptr(hel), _ptr(col)), "bg_generate")


def bg_colour_rule(col) -> bool:
    """Host-only: rule g8 for one event, col[n][2] in {1,2,3}."""
    import numpy as np
    c = np.ascontiguousarray(col, dtype=np.int8)
    rc = load().bg_colour_rule(c.shape[0], _ptr(c))
    if rc < 0:
        raise BgError(rc, "bg_colour_rule")
    return bool(rc)


def bg_eval_host(ctx, N: int, mom, hel, col, out) -> None:
    """Host buffers (numpy arrays or pinned torch CPU tensors), copies included."""
    _check(load().bg_eval_host(ctx, N, _ptr(mom), _ptr(hel), _ptr(col), _ptr(out)), "bg_eval_host")


def bg_reserve(ctx, N: int) -> None:
    _check(load().bg_reserve(ctx, N), "bg_reserve")


def bg_scratch_bytes(ctx, N: int) -> int:
    return int(load().bg_scratch_bytes(ctx, N))


def bg_current_bytes_per_event(ctx) -> int:
    return int(load().bg_current_bytes_per_event(ctx))


def bg_set_option(ctx, key: int, value: int) -> None:
    _check(load().bg_set_option(ctx, key, value), "bg_set_option")


def bg_colour_matrix(ctx, n: int):
    import math
    import numpy as np
    m = math.factorial(n - 2)
    C = np.empty((m, m))
    _check(load().bg_colour_matrix(ctx, _ptr(C)), "bg_colour_matrix")
    return C


def bg_build_colour_matrix(n: int):
    import math
    import numpy as np
    if not 4 <= n <= 8:
        raise BgError(BG_EINVAL, "bg_build_colour_matrix")
    m = math.factorial(n - 2)
    C = np.empty((m, m))
    _check(load().bg_build_colour_matrix(n, _ptr(C)), "bg_build_colour_matrix")
    return C


def bg_last_launch_count(ctx) -> int:
    return int(load().bg_last_launch_count(ctx))


def bg_last_kernel_name(ctx) -> str:
    return load().bg_last_kernel_name(ctx).decode()


def bg_last_kernel_ms(ctx) -> float:
    v = ctypes.c_double()
    _check(load().bg_last_kernel_ms(ctx, ctypes.byref(v)), "bg_last_kernel_ms")
    return v.value


def bg_last_refined(ctx):
    """(events re-evaluated in double-double by the most recent bg_eval, device ms of that re-evaluation)."""
    k, ms = ctypes.c_longlong(), ctypes.c_double()
    _check(load().bg_last_refined(ctx, ctypes.byref(k), ctypes.byref(ms)), "bg_last_refined")
    return int(k.value), ms.value


def bg_last_twin(ctx) -> int:
    """Events of the most recent bg_eval that went through the second (rotated-frame FP64) stage of the cascade."""
    k = ctypes.c_longlong()
    _check(load().bg_last_twin(ctx, ctypes.byref(k)), "bg_last_twin")
    return int(k.value)


def bg_class_program_stats(n: int, lanes: int, counts):
    """Host-only: (valid, vertex_ops, steps, state_bytes, closure_code) of the class program for a colour multiset."""
    import numpy as np
    c = np.ascontiguousarray(counts, dtype=np.int32)
    out = np.zeros(5, dtype=np.int64)
    _check(load().bg_class_program_stats(n, lanes, _ptr(c), _ptr(out)), "bg_class_program_stats")
    return tuple(int(x) for x in out)


def bg_comc_program_stats(n: int, lanes: int, counts):
    """Host-only: (valid, vertex_ops, steps, state_bytes, orderings) of the CO_MC program for a colour multiset."""
    import numpy as np
    c = np.ascontiguousarray(counts, dtype=np.int32)
    out = np.zeros(5, dtype=np.int64)
    _check(load().bg_comc_program_stats(n, lanes, _ptr(c), _ptr(out)), "bg_comc_program_stats")
    return tuple(int(x) for x in out)


def bg_destroy(ctx) -> None:
    _check(load().bg_destroy(ctx), "bg_destroy")


def bg_fp64_peak_probe(iterations: int = 1 << 16) -> float:
    v = ctypes.c_double()
    _check(load().bg_fp64_peak_probe(iterations, ctypes.byref(v)), "bg_fp64_peak_probe")
    return v.value


def bg_colour_form_probe(n: int, E: int, iterations: int = 5, return_data: bool = False):
    """Step a7 alone: (ms per pass with DFMA row dots, ms per pass with mma.sync.m8n8k4.f64, max relative difference)
    [+ amplitudes x[E][2][(n-2)!] and tensor-path results w[E] when return_data]."""
    import math
    import numpy as np
    a, b, d = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    x = w = None
    if return_data:
        x = np.empty((E, 2, math.factorial(n - 2)))
        w = np.empty(E)
    _check(load().bg_colour_form_probe(n, E, iterations, ctypes.byref(a), ctypes.byref(b), ctypes.byref(d), _ptr(x), _ptr(w)),
           "bg_colour_form_probe")
    return (a.value, b.value, d.value) + ((x, w) if return_data else ())


def bg_static_setup() -> None:
    """Resolve the device address of the static scratch array for the current device (once per device)."""
    _check(load().bg_static_setup(), "bg_static_setup")


def bg_static_max_events(n: int) -> int:
    rc = int(load().bg_static_max_events(n))
    if rc < 0:
        raise BgError(rc, "bg_static_max_events")
    return rc


def bg_eval_static(stream, n: int, N: int, mom, hel, col, out) -> None:
    """The no-allocation entry point: CDBG, given helicities and colours, FP64 thread-per-event kernel with its scratch
    in a fixed device array; N <= bg_static_max_events(n), else BgError(BG_ELIMIT).  Device pointers / CUDA tensors."""
    s = ctypes.c_void_p(int(stream)) if stream else None
    _check(load().bg_eval_static(s, n, N, _ptr(mom), _ptr(hel), _ptr(col), _ptr(out)), "bg_eval_static")
