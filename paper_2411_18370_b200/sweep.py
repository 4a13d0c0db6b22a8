"""BASELINE.json configs[4]: the scaling sweep.  `python -m paper_2411_18370_b200.sweep [--max-templates 1e10]`

For every size of sweep A (bank size: n_sft, band width and sky grid grow together, 1e6 .. 1e10
templates) and sweep B (n_sft at a fixed 1 Hz band) it builds the isolated all-sky workload of
config 2 at that size, runs the hot path (ft_eval bind + ft_topk_per_band) with the fused selection
and with the full write-out selection, checks that both return the same candidates, and prints one
JSON line per size: evals/s (fused and full write-out), the statistic kernels' device time, the
fraction of the gather roofline (4 B per evaluation over the measured HBM bandwidth, north_star) and
of the shared-memory roofline (128 B/clk/SM) that binds the tile kernel.  One GPU, no oracle.
"""
from __future__ import annotations

import argparse
import json
import os
import time

import numpy as np

from . import binding as B
from . import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_size(tag, n_sft, band_hz, n_sky, reps, full_writeout, dev, hbm_gbs):
    import torch
    wl = W.config5(n_sft, band_hz, n_sky)
    g = wl.grid
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    P = torch.from_numpy(wl.P).to(dev)
    ctx = B.Context(P, wl.t_mid, wl.vel, wl.w, wl.f_min, wl.df)
    evals = g.n_templates * wl.n_sft
    out = {"sweep": tag, "n_sft": n_sft, "band_hz": band_hz, "n_sky": n_sky, "n_f0": g.n_f0,
           "n_templates": g.n_templates, "evals": evals, "spectrogram_mb": wl.P.nbytes / 1e6}

    def timed(fused):
        ctx.set_option(B.FT_OPT_FUSED_TOPK, fused)
        best, kern, cands = None, None, None
        for r in range(reps + 1):          # first repetition is the warm-up
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ctx.eval(g, "power", wl.rho_th)
            cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)   # synchronises
            dt = time.perf_counter() - t0
            if r > 0 and (best is None or dt < best):
                best, kern = dt, ctx.counters()["last_kernel_ms"]
        return best, kern, cands

    t_f, k_f, c_f = timed(1)
    out.update(kernel=ctx.describe(), fused_s=t_f, fused_evals_per_s=evals / t_f, fused_kernel_ms=k_f,
               gather_roofline_frac=4.0 * evals / (k_f * 1e-3) / 1e9 / hbm_gbs,
               smem_roofline_frac=4.0 * evals / (k_f * 1e-3) / (128.0 * 148 * 1.965e9))
    if full_writeout:
        t_u, k_u, c_u = timed(0)
        out.update(writeout_s=t_u, writeout_evals_per_s=evals / t_u, writeout_kernel_ms=k_u,
                   fused_over_writeout=t_u / t_f,
                   same_candidates=bool(np.array_equal(c_f["idx"], c_u["idx"]) and
                                        np.array_equal(c_f["power"], c_u["power"])))
    ctx.close()
    return out


def run_bank(n, cfg, reps, dev):
    """Unstructured bank of n random templates on config cfg's spectrogram: K1."""
    import torch
    wl = W.by_id(cfg)
    tl = W.random_bank(wl, n)
    P = torch.from_numpy(wl.P).to(dev)
    w = torch.from_numpy(wl.w).to(dev) if wl.per_bin_weights else wl.w
    ctx = B.Context(P, wl.t_mid, wl.vel, w, wl.f_min, wl.df)
    t = torch.from_numpy(tl.view(np.float64).reshape(-1, 8).copy()).to(dev)
    out = torch.empty(n, dtype=torch.float32, device=dev)
    best = None
    for r in range(reps + 1):
        ctx.eval_templates(t, wl.grid.t_ref, "power", wl.rho_th, out, None)   # synchronises
        ms = ctx.counters()["last_kernel_ms"]
        if r > 0 and (best is None or ms < best):
            best = ms
    evals = n * wl.n_sft
    ctx.close()
    return {"bank": "random", "config": cfg, "n_templates": n, "n_sft": wl.n_sft, "evals": evals,
            "kernel_ms": best, "evals_per_s": evals / (best * 1e-3), "kernel": "K1 ft_list_kernel (fp64 per evaluation)"}


def main():
    import torch
    ap = argparse.ArgumentParser()
    ap.add_argument("--bank", type=int, default=0, help="also time an unstructured bank of this many templates (configs 2, 3)")
    ap.add_argument("--max-templates", type=float, default=1.2e9)
    ap.add_argument("--min-templates", type=float, default=0.0)
    ap.add_argument("--reps", type=int, default=2)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("sweep: no CUDA device; the product path has no CPU fallback")
    dev = torch.device("cuda:0")
    try:
        hbm = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except OSError:
        hbm = 6650.0
    if args.bank:
        for cfg in (2, 3):
            print(json.dumps(run_bank(args.bank, cfg, args.reps, dev)), flush=True)
    for tag, sizes in (("A", W.SWEEP_A), ("B", W.SWEEP_B)):
        for n_sft, band_hz, n_sky in sizes:
            n_templates = n_sky * 5 * int(round(band_hz * 1800))
            if n_templates > args.max_templates or n_templates < args.min_templates:
                continue
            print(json.dumps(run_size(tag, n_sft, band_hz, n_sky, args.reps, n_templates <= 2e9, dev, hbm)),
                  flush=True)


if __name__ == "__main__":
    main()
