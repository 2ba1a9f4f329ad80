"""Helpers for the -m gpu tests: run the CUDA path through the C-ABI binding on torch device buffers."""
import numpy as np


def gpu_eval(ev, mode, kernel=0, host=False, scratch_limit=None, lanes=None, smem_limit=None, precision=None,
             flag_threshold=None, flag_twin=None, frame=None):
    """ev: workload.Events (AoS numpy).  Returns out[N] (numpy) and the kernel name used."""
    import torch
    import paper_2106_06507_b200 as bg
    from paper_2106_06507_b200 import workload as wl
    N, n = ev.N, ev.n
    mom = wl.to_soa(mom=ev.mom)
    hel = None if (mode & bg.BG_HEL_SUM) or ev.hel is None else wl.to_soa(hel=ev.hel)
    col = None if not (mode & bg.BG_COL_GIVEN) else wl.to_soa(col=ev.col)
    ctx = bg.bg_init(n, mode)
    try:
        if kernel:
            bg.bg_set_option(ctx, bg.BG_OPT_KERNEL, kernel)
        if lanes is not None:
            try:
                bg.bg_set_option(ctx, bg.BG_OPT_LANES, lanes)
            except bg.BgError as e:
                if e.code == bg.BG_EUNSUPPORTED:
                    import pytest
                    pytest.skip(f"{lanes} lanes per event: one warp's state exceeds shared memory for n={n}")
                raise
        if smem_limit is not None:
            bg.bg_set_option(ctx, bg.BG_OPT_SMEM_LIMIT, smem_limit)
        if precision is not None:
            bg.bg_set_option(ctx, bg.BG_OPT_PRECISION, precision)
        if flag_threshold is not None:
            bg.bg_set_option(ctx, bg.BG_OPT_FLAG_THRESHOLD, flag_threshold)
        if flag_twin is not None:
            bg.bg_set_option(ctx, bg.BG_OPT_FLAG_TWIN, flag_twin)
        if frame is not None:
            bg.bg_set_option(ctx, bg.BG_OPT_FRAME, frame)
        if scratch_limit:
            bg.bg_set_option(ctx, bg.BG_OPT_SCRATCH_LIMIT, scratch_limit)
        if host:
            out = np.full(N, np.nan)
            bg.bg_eval_host(ctx, N, mom, hel, col, out)
        else:
            dev = torch.device("cuda:0")
            d_mom = torch.from_numpy(mom).to(dev)
            d_hel = None if hel is None else torch.from_numpy(hel).to(dev)
            d_col = None if col is None else torch.from_numpy(col).to(dev)
            d_out = torch.full((max(N, 1),), float("nan"), dtype=torch.float64, device=dev)
            stream = torch.cuda.current_stream().cuda_stream
            bg.bg_reserve(ctx, N)
            bg.bg_eval(ctx, stream, N, d_mom, d_hel, d_col, d_out)
            torch.cuda.synchronize()
            out = d_out[:N].cpu().numpy()
        name = bg.bg_last_kernel_name(ctx)
    finally:
        bg.bg_destroy(ctx)
    return out, name


def rel_err(x, truth):
    truth = np.asarray(truth)
    return np.abs(np.asarray(x) - truth) / np.abs(truth)
