"""CPU-side checks of the boundary: libbg.so loads and exports every function include/bg.h declares, error
reporting works without a device, and the host-built colour matrix (Eq. 17) equals the oracle's."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bg():
    from paper_2106_06507_b200 import build as b
    b.build()
    import paper_2106_06507_b200 as bg
    bg.load()
    return bg


def header_functions():
    src = open(os.path.join(ROOT, "include", "bg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bg_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(bg):
    names = header_functions()
    assert len(names) >= 12
    lib = ctypes.CDLL(bg.binding.LIB_PATH)
    for name in names:
        assert hasattr(lib, name), name
    assert set(names) == set(bg.binding.EXPORTS)


def test_strerror_and_modes(bg):
    assert bg.bg_strerror(0) == "ok"
    for code in (-1, -2, -3, -4, -99):
        assert isinstance(bg.bg_strerror(code), str) and bg.bg_strerror(code)
    assert bg.BG_CDBG_GIVEN == 0x222 and bg.BG_COBG_HELSUM_FULLCOLOR == 0x111
    assert bg.BG_COBG_HELGIVEN_FULLCOLOR == 0x121 and bg.BG_COMC_GIVEN == 0x221


def test_init_argument_errors_without_touching_kernels(bg):
    with pytest.raises(bg.BgError) as e:
        bg.bg_init(3, bg.BG_CDBG_GIVEN)
    assert e.value.code == bg.BG_EINVAL
    with pytest.raises(bg.BgError) as e:
        bg.bg_init(13, bg.BG_CDBG_GIVEN)
    assert e.value.code == bg.BG_EINVAL
    with pytest.raises(bg.BgError) as e:
        bg.bg_init(10, bg.BG_COMC_GIVEN)                                       # CO_MC: n <= 9
    assert e.value.code == bg.BG_EUNSUPPORTED
    with pytest.raises(bg.BgError) as e:
        bg.bg_init(6, bg.BG_REC_COBG | bg.BG_HEL_SUM | bg.BG_COL_GIVEN)       # not a combination the library has
    assert e.value.code == bg.BG_EUNSUPPORTED
    with pytest.raises(bg.BgError) as e:
        bg.bg_init(9, bg.BG_COBG_HELGIVEN_FULLCOLOR)                           # colour matrix too large
    assert e.value.code == bg.BG_EUNSUPPORTED


def test_no_silent_cpu_fallback(bg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(bg.BgError) as e:
        bg.bg_init(6, bg.BG_CDBG_GIVEN)
    assert e.value.code == bg.BG_ECUDA


@pytest.mark.parametrize("n", [4, 5, 6, 7])
def test_host_colour_matrix_equals_oracle(bg, oracle, n):
    C = bg.bg_build_colour_matrix(n)
    assert np.array_equal(C, oracle.colour_matrix(n))


def test_host_colour_matrix_n8_properties(bg):
    C = bg.bg_build_colour_matrix(8)
    assert C.shape == (720, 720) and np.array_equal(C, C.T)
    assert np.all(np.diag(C) == 6 ** 6 * 8)
    assert np.all(C == np.rint(C))
    assert np.linalg.eigvalsh(C).min() > -1e-6 * C[0, 0]
    # C_{sigma sigma'} depends only on sigma^-1 sigma' (relabelling the summed colours): every row is a permutation of
    # the first, checked here on a sample of rows against explicitly composed permutations
    import itertools
    perms = list(itertools.permutations(range(6)))
    index = {p: i for i, p in enumerate(perms)}
    for s in (1, 17, 333, 719):
        inv = np.argsort(perms[s])
        for t in (0, 5, 100, 718):
            rel = tuple(int(inv[perms[t][i]]) for i in range(6))
            assert C[s, t] == C[0, index[rel]]
