"""Validation campaign of the default precision path on fresh seeds (not a pytest file; needs a B200):

    python tests/validate_precision.py

For BG_CDBG_GIVEN n = 4..12 and BG_COBG_HELGIVEN_FULLCOLOR n = 5..8 it draws events on the device (bg_generate, streams
7000 + n, seeds 101..), evaluates them with the default path, with the FP64 kernels alone and with every event in
double-double (the reference: within 1e-14 of the long-double oracle on the events checked), and prints
per (mode, n) the number of events over 1e-11, the worst error and the shares of the second and third stage.
profiles/r02_precision_validation.txt is its output at the end of round 2."""
import sys, os
import numpy as np, torch
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_2106_06507_b200 as bg
dev = torch.device("cuda:0")
stream = torch.cuda.current_stream().cuda_stream
def campaign(mode, n, logN, seeds):
    N = 1 << logN
    cdbg = mode == bg.BG_CDBG_GIVEN
    d_mom = torch.empty((n * 4, N), dtype=torch.float64, device=dev)
    d_hel = torch.empty((n, N), dtype=torch.int8, device=dev)
    d_col = torch.empty((n * 2, N), dtype=torch.int8, device=dev) if cdbg else None
    ctx_t = bg.bg_init(n, mode); bg.bg_set_option(ctx_t, bg.BG_OPT_PRECISION, 2); bg.bg_set_option(ctx_t, bg.BG_OPT_FLAG_THRESHOLD, 1); bg.bg_set_option(ctx_t, bg.BG_OPT_FLAG_TWIN, 1)
    ctx = bg.bg_init(n, mode); bg.bg_set_option(ctx, bg.BG_OPT_PRECISION, 2)
    ctx0 = bg.bg_init(n, mode); bg.bg_set_option(ctx0, bg.BG_OPT_PRECISION, 0)
    t = torch.zeros(N, dtype=torch.float64, device=dev); w = torch.zeros_like(t); w0 = torch.zeros_like(t)
    tot = 0; over = 0; worst = 0.0; over0 = 0; worst0 = 0.0; dd = 0; tw = 0; over_list = []
    for seed in seeds:
        bg.bg_generate(stream, n, N, seed, 7000 + n, 0, 1000.0, 20.0, 0.4, True, d_mom, d_hel, d_col)
        bg.bg_eval(ctx_t, stream, N, d_mom, d_hel, d_col, t)
        bg.bg_eval(ctx, stream, N, d_mom, d_hel, d_col, w)
        bg.bg_eval(ctx0, stream, N, d_mom, d_hel, d_col, w0)
        torch.cuda.synchronize()
        dd += bg.bg_last_refined(ctx)[0]; tw += bg.bg_last_twin(ctx)
        ok = t > 0
        e = (torch.abs(w - t) / t)[ok]; e0 = (torch.abs(w0 - t) / t)[ok]
        tot += int(ok.sum()); k = int((e > 1e-11).sum()); over += k; worst = max(worst, float(e.max()))
        over0 += int((e0 > 1e-11).sum()); worst0 = max(worst0, float(e0.max()))
        if k: over_list += [f"{x:.2e}" for x in e[e > 1e-11].cpu().numpy()]
    for c in (ctx_t, ctx, ctx0): bg.bg_destroy(c)
    print(f"{'CDBG' if cdbg else 'COBG'} n={n}: {tot} events ({len(seeds)} x 2^{logN}); default path: {over} over 1e-11 {over_list}, worst {worst:.2e}; second FP64 {tw/tot*100:.2f} %, double-double {dd/tot*100:.2f} %; FP64 alone: {over0} over 1e-11, worst {worst0:.2e}", flush=True)
C, O = bg.BG_CDBG_GIVEN, bg.BG_COBG_HELGIVEN_FULLCOLOR
if len(sys.argv) > 1:         # python tests/validate_precision.py cdbg|cobg n log2N seeds
    campaign(C if sys.argv[1] == "cdbg" else O, int(sys.argv[2]), int(sys.argv[3]), range(101, 101 + int(sys.argv[4])))
    sys.exit(0)
campaign(C, 6, 20, range(101, 117)); campaign(C, 5, 20, range(101, 109)); campaign(C, 7, 19, range(101, 109)); campaign(C, 8, 18, range(101, 109))
campaign(C, 9, 17, range(101, 109)); campaign(C, 10, 16, range(101, 105)); campaign(C, 11, 14, range(101, 103)); campaign(C, 12, 13, range(101, 103)); campaign(C, 4, 20, range(101, 105))
campaign(O, 5, 20, range(101, 105)); campaign(O, 6, 19, range(101, 109)); campaign(O, 7, 18, range(101, 109)); campaign(O, 8, 13, range(101, 105))
