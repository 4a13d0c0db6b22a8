"""bench.py — one "step" = one pass of the whole hot path (track -> bin -> gather -> reduce -> fused
per-band top-k) over one synthetic template bank, through the C ABI.

  python bench.py [--gpus N --steps K --warmup W] [--config 2] [--impl reference]

metric: template·SFT evaluations per second (BASELINE.json).  N=1 workload: BASELINE.json
configs[1] (isolated all-sky, O3-like: 4000 SFTs x 1800 f0 x 5 f1 x 20000 sky = 1.8e8 templates).
N>1: every rank evaluates its own 20000-point slice of an N*20000-point sky grid on a replicated
spectrogram (weak scaling, no data-path collective); the per-band candidates of all ranks are
all-gathered (a few KB) and merged.  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2411_18370_b200 import workloads as W  # noqa: E402

METRIC = "template_sft_evals_per_sec"
UNIT = "evals/s"
# dram__bytes_read.sum + dram__bytes_write.sum per statistic launch (profiles/r01_k2_ncu_full.md: the
# spectrogram is read from HBM once per launch, everything else is served from L2 / shared memory)
NCU_TRAFFIC = {2: 31.23e6}
SMEM_BYTES_PER_CLK_SM = 128.0   # B200_MICROARCH "smem crossbar BW 128 B/cyc/SM"
N_SM = 148


def make_workload(args, rank=0, world=1):
    """The rank's shard of the bank (weak scaling: the sky grid grows with the world size; the
    binary config shards its a_p axis).  Returns (workload with the local grid, index offset)."""
    from paper_2411_18370_b200 import sharding as S
    kw = {"n_sft": args.n_sft} if args.n_sft else {}
    if args.config == 2:
        wl = W.config2(n_sky=(args.n_sky or 20000) * world, **kw)
    elif args.config == 3:
        wl = W.config3(**kw)
    elif args.config == 4:
        wl = W.config4(n_sky=(args.n_sky or 5000) * world, **kw)
    else:
        wl = W.config1()
    off = 0
    if world > 1:
        g, off = S.shard_grid(wl.grid, rank, world)
        assert g is not None, "more ranks than entries on the sharded axis"
        wl.grid = g
    return wl, off


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for j, n in enumerate(names) if any(len(r) >= 7 and r[3 + j] == "Active" for r in self.rows)]
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def oracle_sample(wl, seconds=15.0):
    """Time the oracle, as it stands, on a bounded contiguous sample of the workload's bank."""
    from oracle import ft_oracle as fo
    o = fo.Oracle(wl)
    n_f0 = wl.grid.n_f0
    probe = min(o.n_templates, max(n_f0, 8 * n_f0))
    t0 = time.perf_counter()
    o.eval_range(0, probe)
    dt = max(time.perf_counter() - t0, 1e-6)
    n = int(min(o.n_templates, max(probe, probe * seconds / dt)))
    n = max(n_f0, n // n_f0 * n_f0)
    t0 = time.perf_counter()
    power, count, _, _ = o.eval_range(0, n)
    bpb = int(round(wl.band_width / wl.grid.df0))
    fo.topk_per_band(power if wl.stat != "hough" else count, n_f0, bpb, wl.k)
    dt = time.perf_counter() - t0
    return {"value": n * wl.n_sft / dt, "unit": UNIT, "cores": fo.num_threads(), "kind": "oracle",
            "sample": f"first {n} templates ({n // n_f0} outer points x {n_f0} f0) x {wl.n_sft} SFTs + per-band top-{wl.k}, {dt:.1f} s"}, dt


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores (rank 0 only), a bounded sample per step."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    wl, _ = make_workload(args)
    per_step = 8.0
    for _ in range(args.warmup):
        oracle_sample(wl, seconds=1.0)
    vals, times, last = [], [], None
    for _ in range(args.steps):
        last, dt = oracle_sample(wl, seconds=per_step)
        vals.append(last["value"]); times.append(dt)
    v = float(np.mean(vals))
    last["value"] = v
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(wl, args, 1), "cpu_baseline": last,
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def workload_config(wl, args, world):
    g = wl.grid
    return {"workload": f"BASELINE.json configs[{args.config - 1}] {wl.name}", "n_sft": wl.n_sft,
            "n_bins": wl.n_bins, "n_templates_per_gpu": g.n_templates, "grid": list(map(int, g.dims)),
            "statistic": wl.stat, "band_width_hz": wl.band_width, "k": wl.k,
            "sharding": f"sky axis x{world} (weak)" if world > 1 else "single GPU",
            "l2": "flushed between timed steps (256 MiB write)",
            "injections": "none (noise-only spectrogram; injections need the oracle's track and are test-only)"}


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2411_18370_b200 import binding as B

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    local = local % torch.cuda.device_count()   # (one-GPU boxes: --dist-backend gloo runs every rank on cuda:0)
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    on_dev = args.dist_backend == "nccl"
    if world > 1:
        if on_dev:
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(args.dist_backend)
    wl, idx_off = make_workload(args, rank, world)
    from paper_2411_18370_b200 import sharding as S
    g = wl.grid
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    stream = torch.cuda.current_stream(dev)
    P_host = torch.from_numpy(np.ascontiguousarray(wl.P)).pin_memory()
    w_host = torch.from_numpy(np.ascontiguousarray(wl.w)).pin_memory() if wl.per_bin_weights else None
    P_dev = P_host.to(dev)
    w_arg = w_host.to(dev) if wl.per_bin_weights else wl.w
    ctx = B.Context(P_dev, wl.t_mid, wl.vel, w_arg, wl.f_min, wl.df, stream)
    ctx.set_option(B.FT_OPT_KERNEL, args.kernel)
    ctx.set_option(B.FT_OPT_FUSED_TOPK, args.fused)
    ctx.set_option(B.FT_OPT_POINTS_PER_CTA, args.ppc)
    ctx.set_option(B.FT_OPT_F0_TILES, args.tiles)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    evals = g.n_templates * wl.n_sft

    def step(c):
        c.eval(g, wl.stat, wl.rho_th)                      # bind grid (+ fold weights / threshold bit)
        cands = c.topk_per_band(wl.band_width, wl.k, n_bands)   # evaluate + fused selection; syncs
        if world > 1:  # KBs of records: all-gather + merge under the same total order
            cands = S.merge_candidates(S.all_gather_candidates(S.to_global(cands, idx_off), dev if on_dev else None), wl.k,
                                       by_count=(wl.stat == "hough"))
        return cands

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step(ctx)
    c0 = ctx.counters()
    sampler = ClockSampler(local); sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms, kern_n = [], []
    barrier()
    for s in range(args.steps):
        flush.fill_(s & 255)                                # flush L2 between timed steps
        ev[s][0].record(stream)
        step(ctx)
        ev[s][1].record(stream)
        cs = ctx.counters()
        kern_ms.append(cs["last_kernel_ms"]); kern_n.append(cs["stat_launches"])
    barrier()
    clocks = sampler.stop()
    c1 = ctx.counters()
    ms = np.array([a.elapsed_time(b) for a, b in ev])
    tot = torch.tensor([float(ms.sum())], device=dev if on_dev else "cpu")
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.MAX)
    total_ms = float(tot.item())
    value = evals * world * args.steps / (total_ms * 1e-3)

    # end to end through the C ABI from HOST buffers: H2D of the spectrogram (+ per-bin weights),
    # ft_create, ft_eval, ft_topk_per_band, candidates back on the host
    e2e_ms = []
    for s in range(max(2, min(args.steps, 5)) + 1):
        barrier()
        t0 = time.perf_counter()
        Pd = torch.empty_like(P_dev); Pd.copy_(P_host, non_blocking=True)
        wa = wl.w
        if wl.per_bin_weights:
            wa = torch.empty_like(w_arg); wa.copy_(w_host, non_blocking=True)
        c2 = B.Context(Pd, wl.t_mid, wl.vel, wa, wl.f_min, wl.df, stream)
        c2.set_option(B.FT_OPT_KERNEL, args.kernel); c2.set_option(B.FT_OPT_FUSED_TOPK, args.fused)
        c2.set_option(B.FT_OPT_POINTS_PER_CTA, args.ppc); c2.set_option(B.FT_OPT_F0_TILES, args.tiles)
        cands = step(c2)
        barrier()
        if s > 0:
            e2e_ms.append(1e3 * (time.perf_counter() - t0))
        c2.close()
    e2e_t = torch.tensor([float(np.mean(e2e_ms))], device=dev if on_dev else "cpu")
    if world > 1:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    h2d = P_host.numel() * 4 * (2 if wl.per_bin_weights else 1) + wl.n_sft * (8 + 24 + 4) + g.sky.size * 8
    d2h = int(cands.nbytes)

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        k_ms = float(np.mean(kern_ms))                     # statistic-kernel device time per step
        n_launch = float(np.mean(kern_n))                  # statistic-kernel launches per step
        # per launch: 4 B x (evals / n_launch) over (k_ms / n_launch) -- algorithmic gather bytes
        achieved = 4.0 * evals / (k_ms * 1e-3) / 1e9
        traffic = args.traffic if args.traffic is not None else NCU_TRAFFIC.get(args.config)
        sm_mhz = clocks.get("sm_mhz") or 1965.0
        smem_peak = SMEM_BYTES_PER_CLK_SM * N_SM * sm_mhz * 1e6 / 1e9
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": workload_config(wl, args, world),
            "templates_per_sec": value / wl.n_sft,
            "gpu_launches": int(c1["kernel_launches"] - c0["kernel_launches"]),
            "clocks": clocks,
            "e2e": {"value": evals * world / (float(e2e_t.item()) * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": d2h},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                         "frac": achieved / hbm_peak, "traffic": traffic,
                         "kernel": "ft_tile_kernel (K2) / ft_generic_kernel (K0): the statistic launches of ft_topk_per_band, CUDA events on the library's stream around each launch, summed per step, mean over timed steps",
                         "kernel_ms": k_ms, "launches_per_step": n_launch,
                         "algorithmic_bytes_per_launch": 4.0 * evals / max(n_launch, 1.0),
                         "share_of_step": k_ms / (total_ms / args.steps),
                         "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks else "fallback 6650 GB/s (of fallback)",
                         "note": "north_star gather roofline: 4 B per template·SFT eval over HBM/L2 bandwidth; strips staged once in shared memory are re-read by many templates, so frac can exceed 1 — see tight",
                         "tight": {"bound": "smem", "peak": smem_peak, "unit": "GB/s", "frac": achieved / smem_peak,
                                   "how": f"128 B/clk/SM x 148 SMs x {sm_mhz:.0f} MHz (median SM clock during the timed region)"}},
            "counters": {k: c1[k] for k in ("near_ties", "appended", "refined", "refine_fallbacks")},
            "kernel_geometry": ctx.describe(),
        }
        if not args.no_cpu_baseline and world == 1:
            out["cpu_baseline"], _ = oracle_sample(wl, seconds=args.cpu_seconds)
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4])
    ap.add_argument("--n-sky", type=int, default=0)
    ap.add_argument("--n-sft", type=int, default=0)
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 generic, 2 tile")
    ap.add_argument("--fused", type=int, default=1)
    ap.add_argument("--tiles", type=int, default=0, help="f0 tiles (0 = library default)")
    ap.add_argument("--ppc", type=int, default=0, help="outer points per CTA (0 = library default)")
    ap.add_argument("--traffic", type=float, default=None, help="ncu dram bytes per launch (from profiles/)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="gloo: exercise the N>1 path with every rank on one GPU (testing only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
