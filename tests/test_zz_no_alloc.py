"""bg_eval_static, the no-allocation entry point (include/bg.h): the thread-per-event CDBG kernel with its scratch in a
fixed file-scope device array.  Collected last on purpose (the suite runs with pytest -x).

Checked against the existing path - bg_eval of a BG_CDBG_GIVEN context under BG_OPT_KERNEL = 1, the same kernel with
cudaMalloc'ed scratch - at the 1e-11 of the parity tests (the arithmetic is the same, so the bits agree too), on two
calls in a row that share the array, and against the long-double oracle at the FP64 bar of the other FP64-only kernels."""
import numpy as np
import pytest

from gpu_util import gpu_eval, rel_err
from test_gpu_parity import check_cdbg_fp64


@pytest.fixture(scope="module")
def bg():
    import paper_2106_06507_b200 as bg
    bg.load()
    return bg


def test_static_limits_are_host_side(bg):
    """bg_static_max_events needs no GPU: BG_STATIC_SCRATCH_BYTES / (2^(n-1) x 513 bytes per event)."""
    assert bg.BG_STATIC_SCRATCH_BYTES == 32 << 20
    for n in range(4, 13):
        assert bg.bg_static_max_events(n) == (32 << 20) // ((1 << (n - 1)) * 513)
    assert bg.bg_static_max_events(6) == 2044 and bg.bg_static_max_events(12) == 31
    for n in (3, 13):
        with pytest.raises(bg.BgError) as e:
            bg.bg_static_max_events(n)
        assert e.value.code == bg.BG_EINVAL
    assert "bg_static_max_events" in bg.bg_strerror(bg.BG_ELIMIT)


def _to_device(wl, ev):
    import torch
    dev = torch.device("cuda:0")
    return tuple(torch.from_numpy(a).to(dev) for a in (wl.to_soa(mom=ev.mom), wl.to_soa(hel=ev.hel), wl.to_soa(col=ev.col)))


def _static_eval(bg, ev, inputs, d_out):
    import torch
    bg.bg_eval_static(torch.cuda.current_stream().cuda_stream, ev.n, ev.N, *inputs, d_out)


@pytest.mark.gpu
@pytest.mark.parametrize("n", [6, 8, 12])
def test_static_entry_point_matches_existing_path_twice(bg, oracle, wl, n):
    import torch
    cap = bg.bg_static_max_events(n)
    first = wl.config_events(4, N=cap, n=n)                        # fills the array to its limit
    second = wl.config_events(4, N=max(cap // 2 - 3, 1), n=n, seed=7)   # then a ragged batch over the leftovers of the first
    bg.bg_static_setup()
    bg.bg_static_setup()                                           # idempotent
    dev = torch.device("cuda:0")
    outs = [torch.full((ev.N,), float("nan"), dtype=torch.float64, device=dev) for ev in (first, second)]
    inputs = [_to_device(wl, ev) for ev in (first, second)]
    _static_eval(bg, first, inputs[0], outs[0])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    _static_eval(bg, second, inputs[1], outs[1])                   # second call in a row, same stream, same array
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "bg_eval_static changed the amount of free device memory"
    for ev, out in zip((first, second), outs):
        got = out.cpu().numpy()
        ref, name = gpu_eval(ev, bg.BG_CDBG_GIVEN, kernel=1)       # the existing path: same kernel, context-owned scratch
        assert name == "cdbg_generic_kernel"
        assert np.all(np.isfinite(got))
        assert np.all(rel_err(got[ref != 0], ref[ref != 0]) <= 1e-11)
        assert np.array_equal(got == 0, ref == 0)
        assert np.array_equal(got, ref)                            # same arithmetic: the bits agree
        check_cdbg_fp64(oracle, ev, got, max_tail_frac=0.02)


@pytest.mark.gpu
def test_static_entry_point_rejects_what_does_not_fit(bg, wl):
    import torch
    n = 7
    cap = bg.bg_static_max_events(n)
    ev = wl.config_events(4, N=cap + 1, n=n)
    dev = torch.device("cuda:0")
    out = torch.full((ev.N,), -1.0, dtype=torch.float64, device=dev)
    inputs = _to_device(wl, ev)
    with pytest.raises(bg.BgError) as e:
        _static_eval(bg, ev, inputs, out)
    assert e.value.code == bg.BG_ELIMIT
    torch.cuda.synchronize()
    assert bool((out == -1.0).all())                               # nothing was launched
    with pytest.raises(bg.BgError) as e:
        bg.bg_eval_static(0, 3, 8, out, out, out, out)
    assert e.value.code == bg.BG_EINVAL
    with pytest.raises(bg.BgError) as e:
        bg.bg_eval_static(0, n, 8, None, out, out, out)
    assert e.value.code == bg.BG_EINVAL
    bg.bg_eval_static(0, n, 0, None, None, None, None)             # N = 0: no-op
