"""bench.py — one "step" = one pass of the whole hot path (track -> bin -> gather -> reduce -> fused
per-band top-k) over one synthetic template bank, through the C ABI.

  python bench.py [--gpus N --steps K --warmup W] [--config 2] [--impl reference]

metric: template·SFT evaluations per second (BASELINE.json).  N=1 workload: BASELINE.json
configs[1] (isolated all-sky, O3-like: 4000 SFTs x 1800 f0 x 5 f1 x 20000 sky = 1.8e8 templates).
N>1: every rank evaluates its own 20000-point slice of an N*20000-point sky grid on a replicated
spectrogram (weak scaling, no data-path collective); the per-band candidates of all ranks are
all-gathered (a few KB) and merged.  `--gpus N` with N > 1 and no WORLD_SIZE in the environment starts
the N ranks itself (torch.distributed.run on 127.0.0.1).  Prints ONE JSON line (rank 0).

The default run also times, after the headline, the other target configuration (BASELINE.json configs[2],
binary) and configs[3], the packed number-count and one-pass kernels and the unstructured-bank kernel K1
(`extra`), so that every fraction of BASELINE.md §4 can be recomputed from this one line.
`--config 5` runs BASELINE.json configs[4], the scaling sweep (`sweep` in the JSON line).
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import socket
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
SMEM_BYTES_PER_CLK_SM = 128.0   # nominal: B300_MICROARCH "smem crossbar BW 128 B/cyc/SM" (fallback when not measured)
FP64_FMA_PER_CLK_SM = 64.0      # nominal B200 vector fp64 (40 TFLOP/s at 148 SMs x 1.965 GHz / 2)
N_SM = 148
# fp64-pipe cycles per evaluation of K1, in DFMA-equivalents, from ncu sm__pipe_fp64_cycles_active (profiles/r02_k1_*_ncu.md)
K1_FP64_SLOTS = {"isolated": 19.2, "binary": 41.3}


def ncu_traffic(config: int, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on BASELINE config `config`, from the
    committed ncu summary table (profiles/r02_dram_traffic.csv; each row names the capture it comes from)."""
    try:
        with open(os.path.join(ROOT, "profiles", "r02_dram_traffic.csv")) as fh:
            for row in csv.DictReader(fh):
                if int(row["config"]) == config and row["kernel"] == kernel:
                    return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
    except (OSError, KeyError, ValueError):
        pass
    return None


def make_workload(args, rank=0, world=1, config=None):
    """The rank's shard of the bank (weak scaling: the sky grid grows with the world size; the
    binary config shards its a_p axis).  Returns (workload with the local grid, index offset)."""
    from paper_2411_18370_b200 import sharding as S
    config = config or args.config
    kw = {"n_sft": args.n_sft} if args.n_sft else {}
    if config == 2:
        wl = W.config2(n_sky=(args.n_sky or 20000) * world, **kw)
    elif config == 3:
        wl = W.config3(**kw)
    elif config == 4:
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
    per_step = args.cpu_seconds if args.cpu_seconds_set else 8.0
    for _ in range(args.warmup):
        oracle_sample(wl, seconds=min(1.0, per_step))
    vals, times, last = [], [], None
    for _ in range(max(1, args.steps)):
        last, dt = oracle_sample(wl, seconds=per_step)
        vals.append(last["value"]); times.append(dt)
    v = float(np.mean(vals))
    last["value"] = v
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(wl, args, 1, args.config), "cpu_baseline": last,
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def workload_config(wl, args, world, config):
    g = wl.grid
    return {"workload": f"BASELINE.json configs[{config - 1}] {wl.name}", "n_sft": wl.n_sft,
            "n_bins": wl.n_bins, "n_templates_per_gpu": g.n_templates, "grid": list(map(int, g.dims)),
            "statistic": wl.stat, "band_width_hz": wl.band_width, "k": wl.k,
            "sharding": f"sky axis x{world} (weak)" if world > 1 else "single GPU",
            "l2": "flushed between timed steps (256 MiB write)",
            "injections": "none (noise-only spectrogram; injections need the oracle's track and are test-only)"}


class Runner:
    """One workload on the device: context, the hot-path step, device-timed repetitions."""

    def __init__(self, wl, dev, args, stat=None):
        import torch
        from paper_2411_18370_b200 import binding as B
        self.torch, self.B, self.wl, self.dev, self.args = torch, B, wl, dev, args
        self.stat = stat or wl.stat
        g = wl.grid
        self.bpb = int(round(wl.band_width / g.df0)); self.n_bands = -(-g.n_f0 // self.bpb)
        self.stream = torch.cuda.current_stream(dev)
        self.P_host = torch.from_numpy(np.ascontiguousarray(wl.P)).pin_memory()
        self.w_host = torch.from_numpy(np.ascontiguousarray(wl.w)).pin_memory() if wl.per_bin_weights else None
        self.P_dev = self.P_host.to(dev)
        self.w_arg = self.w_host.to(dev) if wl.per_bin_weights else wl.w
        self.ctx = self.make_ctx(self.P_dev, self.w_arg)
        self.evals = g.n_templates * wl.n_sft

    def make_ctx(self, P_dev, w_arg):
        B, args, wl = self.B, self.args, self.wl
        ctx = B.Context(P_dev, wl.t_mid, wl.vel, w_arg, wl.f_min, wl.df, self.stream)
        ctx.set_option(B.FT_OPT_KERNEL, args.kernel)
        ctx.set_option(B.FT_OPT_FUSED_TOPK, args.fused)
        ctx.set_option(B.FT_OPT_POINTS_PER_CTA, args.ppc)
        ctx.set_option(B.FT_OPT_F0_TILES, args.tiles)
        return ctx

    def step(self, ctx=None):
        c = ctx or self.ctx
        c.eval(self.wl.grid, self.stat, self.wl.rho_th)                  # bind grid (+ fold weights / threshold bit)
        return c.topk_per_band(self.wl.band_width, self.wl.k, self.n_bands)   # evaluate + fused selection; syncs

    def full_arrays_step(self):
        """The other kind of step: every statistic of the bank written out (A5), no selection."""
        torch, wl = self.torch, self.wl
        n = wl.grid.n_templates
        op = torch.empty(n, dtype=torch.float32, device=self.dev) if self.stat != "hough" else None
        oc = torch.empty(n, dtype=torch.int32, device=self.dev) if self.stat not in ("power", "whough") else None

        def step(ctx=None):
            (ctx or self.ctx).eval(wl.grid, self.stat, wl.rho_th, op, oc)
            torch.cuda.synchronize()
            return np.zeros(0, dtype=np.uint8)
        return step

    def timed(self, steps, warmup, flush, barrier=lambda: None, step=None):
        """Device-timed steps with an L2 flush between them.  Returns (per-step ms array, statistic-kernel ms per
        step, statistic launches per step)."""
        torch = self.torch
        step = step or self.step
        for _ in range(warmup):
            step()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        kern_ms, kern_n = [], []
        barrier()
        for s in range(steps):
            flush.fill_(s & 255)                                # flush L2 between timed steps
            ev[s][0].record(self.stream)
            step()
            ev[s][1].record(self.stream)
            cs = self.ctx.counters()
            kern_ms.append(cs["last_kernel_ms"]); kern_n.append(cs["stat_launches"])
        barrier()
        ms = np.array([a.elapsed_time(b) for a, b in ev])
        return ms, float(np.mean(kern_ms)), float(np.mean(kern_n))

    def close(self):
        self.ctx.close()


def roofline_block(evals, k_ms, n_launch, step_ms, peaks, measured, sm_mhz, traffic, kernel_note):
    """`bound`: the unit that binds the tile kernel is the shared-memory data pipe (ncu: profiles/r0*_k2_*.md);
    peak = the conflict-free LDS.32 bandwidth ft_measure_peaks measured on this device in this run, else the
    nominal 128 B/clk/SM at the sampled clock.  `gather` is north_star's roofline: the same algorithmic bytes
    over the measured HBM copy bandwidth (a strip staged once in shared memory serves every template of the
    CTA, so that fraction exceeds 1)."""
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    achieved = 4.0 * evals / (k_ms * 1e-3) / 1e9
    nominal = SMEM_BYTES_PER_CLK_SM * N_SM * sm_mhz * 1e6 / 1e9
    smem_peak = float(measured["smem_gbs"]) if measured else nominal
    return {"bound": "smem", "achieved": achieved, "peak": smem_peak, "unit": "GB/s", "frac": achieved / smem_peak,
            "traffic": traffic,
            "peak_source": ("ft_measure_peaks: conflict-free LDS.32 from every SM, this device, this run (of measured)" if measured
                            else f"nominal 128 B/clk/SM x 148 SMs x {sm_mhz:.0f} MHz (of nominal)"),
            "peak_nominal": nominal, "frac_of_nominal": achieved / nominal,
            "kernel": kernel_note, "kernel_ms": k_ms, "launches_per_step": n_launch,
            "algorithmic_bytes_per_launch": 4.0 * evals / max(n_launch, 1.0),
            "algorithmic_bytes_per_eval": 4.0,
            "share_of_step": k_ms / step_ms,
            "gather": {"bound": "hbm", "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                       "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks else "fallback 6650 GB/s (of fallback)",
                       "note": "north_star gather roofline: 4 B per template·SFT evaluation over HBM/L2 bandwidth"}}


def bank_run(args, dev, flush, wl, binary, measured):
    """K1 on a xi-uniform random bank (Eq. A11) over the workload's parameter box, drawn and evaluated on the device
    by one ft_eval_bank call; best of two timed repetitions after a warm-up."""
    r = Runner(wl, dev, args)
    g = wl.grid
    binary = bool(binary and float(np.max(g.a_p)) > 0.0)   # (--only-bank binary on an isolated configuration: isolated bank)
    box = dict(f0_lo=g.f0_start, f0_hi=g.f0_start + (g.n_f0 - 1) * g.df0, f1_lo=g.f1_start, f1_hi=g.f1_start + (g.n_f1 - 1) * g.df1,
               ra_lo=0.0, ra_hi=2 * np.pi, sd_lo=-1.0, sd_hi=1.0,
               ap_lo=float(np.min(g.a_p)) if binary else 0.0, ap_hi=float(np.max(g.a_p)) if binary else 0.0,
               porb_lo=float(np.min(g.P_orb)), porb_hi=float(np.max(g.P_orb)), t_ref=g.t_ref)
    if binary:
        n0 = g.sky[0]
        ra = float(np.arctan2(n0[1], n0[0]) % (2 * np.pi))
        box.update(ra_lo=ra, ra_hi=ra, sd_lo=float(n0[2]), sd_hi=float(n0[2]))
    n = args.bank
    best_ms = None
    for rep in range(3):
        flush.fill_(rep)
        r.ctx.eval_bank(box, 7, 0, n, "power", wl.rho_th)          # synchronises
        ms = r.ctx.counters()["last_kernel_ms"]
        if rep > 0:
            best_ms = ms if best_ms is None else min(best_ms, ms)
    evals = n * wl.n_sft
    fp64_peak = (measured["fp64_gflops"] / 2.0 * 1e9) if measured else FP64_FMA_PER_CLK_SM * N_SM * 1.965e9
    # fp64-pipe slots per evaluation (SASS of k1_chunk)
    instr = K1_FP64_SLOTS["binary" if binary else "isolated"]
    res = {"workload": f"{n} templates uniform in xi (Eq. A11) on the spectrogram of {wl.name}", "kernel": "K1 ft_list_kernel (drawn in registers)",
           "value": evals / (best_ms * 1e-3), "unit": UNIT, "kernel_ms": best_ms,
           "bound": "alu (fp64 pipe)", "fp64_pipe_slots_per_eval": instr,
           "roofline_frac": evals * instr / (best_ms * 1e-3) / fp64_peak,
           "roofline_frac_of_nominal": evals * instr / (best_ms * 1e-3) / (FP64_FMA_PER_CLK_SM * N_SM * 1.965e9),
           "peak": fp64_peak, "peak_unit": "fp64 instr/s",
           "peak_source": "ft_measure_peaks DFMA rate (of measured)" if measured else "nominal 64 DFMA/clk/SM (of nominal)"}
    if not binary and not wl.per_bin_weights:
        # the paper's per-box step on a random bank, end to end (Eq. 36): sky-dependent weights
        # (Eq. 4-5) per template, both statistics, weighted-count floor mu + 3 sigma, loudest by z -- ft_eval_bank_veto
        r.ctx.set_antenna(*W.antenna_geometry(wl))
        p_hit = float(np.exp(-wl.rho_th))
        n_eff = wl.n_sft      # (sum w = 1 per sky point; sum w^2 ~ 1 / n_sft: the floor of a uniform-weight bank)
        wfloor = p_hit + 3.0 * np.sqrt(p_hit * (1.0 - p_hit) / n_eff)
        veto_ms = None
        for rep in range(3):
            flush.fill_(rep)
            best, _ = r.ctx.eval_bank_veto(box, 7, 0, n, wl.rho_th, wfloor, True)
            ms = r.ctx.counters()["last_kernel_ms"]
            if rep > 0:
                veto_ms = ms if veto_ms is None else min(veto_ms, ms)
        res["per_box_procedure"] = {"call": "ft_set_antenna + ft_eval_bank_veto (both statistics, weighted-count floor, loudest by z)",
                                    "value": evals / (veto_ms * 1e-3), "unit": UNIT, "kernel_ms": veto_ms,
                                    "wcount_floor": wfloor, "winner_found": bool(best["idx"] != np.uint64(2 ** 64 - 1)),
                                    "winner_z": float(best["z"])}
        r.ctx.set_antenna(None)
    r.close()
    return res


def sampler_run(wl, dev):
    """the mismatch-distribution sampler on the binary configuration's noise:
    3 signals from the priors of a box with N(Delta lambda) ~ 4e6 (Eq. A10), oversampling 1; templates per second
    INCLUDING their generation -- what the paper's own benchmark counts."""
    from paper_2411_18370_b200 import sampler as S
    g = wl.grid
    n = g.sky[0]
    ra = float(np.arctan2(n[1], n[0]) % (2 * np.pi)); sd = float(n[2])
    f_mid = g.f0_start + 0.5 * g.n_f0 * g.df0
    box = dict(f0_lo=f_mid, f0_hi=f_mid + 0.01, f1_lo=0.0, f1_hi=0.0, ra_lo=ra - 0.25, ra_hi=ra + 0.25,
               sd_lo=max(-1.0, sd - 0.25), sd_hi=min(1.0, sd + 0.25), ap_lo=2.0, ap_hi=10.0,
               porb_lo=15 * 86400.0, porb_hi=25 * 86400.0, t_ref=g.t_ref)
    T_obs = float(wl.t_mid.max() - wl.t_mid.min()) + wl.T_sft
    S.mismatch_samples(wl, box, n_inj=1, oversampling=0.0, seed=40, amp=3.0, T_obs=T_obs, n_bank=100_000, device=dev)   # warm-up
    r = S.mismatch_samples(wl, box, n_inj=3, oversampling=1.0, seed=41, amp=3.0, T_obs=T_obs, device=dev)
    return {"workload": f"mismatch sampler on the noise of {wl.name}: 3 injected signals (amplitude +3 per SFT), box with N = {r['N']:.4g} (Eq. A10), o = 1",
            "kernel": "K1 ft_list_kernel via ft_eval_bank (drawn in registers, loudest of the bank refined in fp64)",
            "n_bank": r["n_bank"], "templates_per_sec_incl_generation": r["bank_templates"] / r["bank_seconds"],
            "value": r["bank_templates"] * wl.n_sft / r["bank_seconds"], "unit": UNIT, "timing": "host clock around the synchronising ft_eval_bank calls",
            "mismatch": [float(x) for x in r["m"]]}


def extra_runs(args, dev, flush, measured, peaks, sm_mhz_of):
    """The other target configuration and the other kernels, two timed steps each (device-timed, L2 flushed)."""
    import torch
    from paper_2411_18370_b200 import binding as B
    out = {}

    def one(tag, wl, config, stat=None, step_kind="topk", traffic_kernel="ft_tile_kernel", prepare=None, step_of=None):
        r = Runner(wl, dev, args, stat=stat)
        if prepare:
            prepare(r)
        step = step_of(r) if step_of else r.full_arrays_step() if step_kind == "full" else r.step
        sampler = ClockSampler(dev.index or 0); sampler.start()
        ms, k_ms, n_launch = r.timed(2, 2, flush, step=step)
        clocks = sampler.stop()
        mhz = clocks.get("sm_mhz") or 1965.0
        rb = roofline_block(r.evals, k_ms, n_launch, float(ms.mean()), peaks, measured, mhz,
                            ncu_traffic(config, traffic_kernel), r.ctx.describe())
        out[tag] = {"workload": f"BASELINE.json configs[{config - 1}] {wl.name}", "statistic": r.stat, "step": step_kind,
                    "value": r.evals / (float(ms.mean()) * 1e-3), "unit": UNIT, "ms_per_step": float(ms.mean()),
                    "kernel_ms": k_ms, "launches_per_step": n_launch,
                    "roofline_frac": rb["frac"], "roofline_frac_of_nominal": rb["frac_of_nominal"],
                    "gather_frac": rb["gather"]["frac"], "traffic": rb["traffic"],
                    "clocks": {"sm_mhz": clocks.get("sm_mhz"), "reasons": clocks.get("reasons")},
                    "kernel_geometry": r.ctx.describe()}
        r.close()

    wl3, _ = make_workload(args, config=3)
    one("cfg3_power_topk", wl3, 3, stat="power")
    one("cfg3_both_topk", wl3, 3, stat="both")
    one("cfg3_both_full_arrays_k2b", wl3, 3, stat="both", step_kind="full", traffic_kernel="ft_tileb_kernel")
    wl4, _ = make_workload(args, config=4)
    one("cfg4_power_topk", wl4, 4)
    del wl4
    wl2, _ = make_workload(args, config=2)
    one("cfg2_count_full_array_k2h", wl2, 2, stat="hough", step_kind="full", traffic_kernel="ft_tile8_kernel")
    # the weighted number count as the statistic; sky-dependent weights (Eq. 4-5) with the paper's
    # post-processing (loudest template per box of sky points x sub-band, ranked by z, Eq. 36); power top-k under the
    # weighted-count veto
    one("cfg2_weighted_count_topk", wl2, 2, stat="whough", step_kind="topk (ranked by the weighted number count)")
    n_pts = wl2.grid.n_templates // wl2.grid.n_f0
    pbox = (np.arange(n_pts, dtype=np.int64) * 16 // n_pts).astype(np.int32)

    def box_step(r):
        def step():
            r.ctx.eval(wl2.grid, "power", wl2.rho_th)
            return r.ctx.topk_per_box(pbox, 16, wl2.band_width, 1, rank_by_z=True)
        return step
    one("cfg2_antenna_weights_loudest_per_box_by_z", wl2, 2, stat="power", step_kind="ft_eval + ft_topk_per_box (16 boxes of sky points x 20 sub-bands, k = 1, by z)",
        traffic_kernel="ft_tilew_kernel", prepare=lambda r: r.ctx.set_antenna(*W.antenna_geometry(wl2)), step_of=box_step)
    p_hit = float(np.exp(-wl2.rho_th)); w2 = np.asarray(wl2.w, dtype=np.float64)
    wfloor = p_hit * w2.sum() + 3.0 * np.sqrt(p_hit * (1.0 - p_hit) * (w2 ** 2).sum())
    one("cfg2_power_topk_weighted_count_veto", wl2, 2, stat="both", step_kind="topk under the weighted number-count floor mu + 3 sigma",
        prepare=lambda r: r.ctx.set_option_f64(B.FT_OPT_WCOUNT_FLOOR, wfloor))
    # K1: a xi-uniform random bank, drawn and evaluated on the device
    out["mismatch_sampler_cfg3"] = sampler_run(wl3, dev)
    out["k1_bank_cfg2_isolated"] = bank_run(args, dev, flush, wl2, False, measured)
    out["k1_bank_cfg3_binary"] = bank_run(args, dev, flush, wl3, True, measured)
    return out


def run_sweep(args, dev, flush, measured, peaks):
    """BASELINE.json configs[4]: sweep A (bank size) and B (n_sft); fused selection vs full write-out."""
    import torch
    from paper_2411_18370_b200 import binding as B
    torch_sync = torch.cuda.synchronize
    rows = []
    for tag, sizes in (("A", W.SWEEP_A), ("B", W.SWEEP_B)):
        for n_sft, band_hz, n_sky in sizes:
            n_templates = n_sky * 5 * int(round(band_hz * 1800))
            if n_templates > args.sweep_max_templates or n_templates < args.sweep_min_templates:
                continue
            wl = W.config5(n_sft, band_hz, n_sky)
            r = Runner(wl, dev, args)
            row = {"sweep": tag, "n_sft": n_sft, "band_hz": band_hz, "n_sky": n_sky, "n_f0": wl.grid.n_f0,
                   "n_templates": wl.grid.n_templates, "evals": r.evals, "spectrogram_mb": wl.P.nbytes / 1e6}
            res = {}
            for fused in ((1, 0) if n_templates <= 2e9 else (1,)):
                r.ctx.set_option(B.FT_OPT_FUSED_TOPK, fused)
                best, kern, cands = None, None, None
                for rep in range(args.sweep_reps + 1):          # first repetition is the warm-up
                    flush.fill_(rep)
                    torch_sync()
                    self_t0 = time.perf_counter()
                    cands = r.step()
                    dt = time.perf_counter() - self_t0
                    if rep > 0 and (best is None or dt < best):
                        best, kern = dt, r.ctx.counters()["last_kernel_ms"]
                res[fused] = (best, kern, cands)
            t_f, k_f, c_f = res[1]
            smem_peak = measured["smem_gbs"] if measured else SMEM_BYTES_PER_CLK_SM * N_SM * 1.965
            row.update(kernel=r.ctx.describe(), fused_s=t_f, fused_evals_per_s=r.evals / t_f, fused_kernel_ms=k_f,
                       gather_roofline_frac=4.0 * r.evals / (k_f * 1e-3) / 1e9 / float(peaks.get("hbm_gbs", 6650.0)),
                       smem_roofline_frac=4.0 * r.evals / (k_f * 1e-3) / 1e9 / smem_peak)
            if 0 in res:
                t_u, k_u, c_u = res[0]
                row.update(writeout_s=t_u, writeout_evals_per_s=r.evals / t_u, writeout_kernel_ms=k_u, fused_over_writeout=t_u / t_f,
                           same_candidates=bool(np.array_equal(c_f["idx"], c_u["idx"]) and np.array_equal(c_f["power"], c_u["power"])))
            r.close()
            rows.append(row)
    return rows


def run_gpu(args):
    import torch
    import torch.distributed as dist

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
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    from paper_2411_18370_b200 import sharding as S

    if args.config == 5:
        wl0 = W.config1()
        r0 = Runner(wl0, dev, args)
        measured = r0.ctx.measure_peaks() if not args.no_peaks else None
        r0.close()
        rows = run_sweep(args, dev, flush, measured, peaks)
        big = max(rows, key=lambda r: r["evals"])
        print(json.dumps({"metric": METRIC, "value": big["fused_evals_per_s"], "unit": UNIT, "n_gpus": 1, "steps": args.sweep_reps,
                          "warmup": 1, "ms_per_step": 1e3 * big["fused_s"], "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": {"workload": "BASELINE.json configs[4] scaling sweep (value: the largest size run)", "timing": "host wall-clock around ft_eval (bind) + ft_topk_per_band (synchronises), best of reps after a warm-up"},
                          "measured_peaks": measured, "sweep": rows}))
        return

    wl, idx_off = make_workload(args, rank, world)
    g = wl.grid
    if args.only_bank:   # K1 alone (the command of profiles/r02_k1_*.md)
        r0 = Runner(wl, dev, args)
        measured = r0.ctx.measure_peaks() if not args.no_peaks else None
        r0.close()
        res = bank_run(args, dev, flush, wl, args.only_bank == "binary", measured)
        print(json.dumps({"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": 1, "steps": 2, "warmup": 1,
                          "ms_per_step": res["kernel_ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                          "dtype": "f64", "data": "synthetic", "config": {"workload": res["workload"]}, "k1": res}))
        return
    r = Runner(wl, dev, args, stat=("both" if args.veto_sigma > 0 else args.stat) or None)
    measured = r.ctx.measure_peaks() if not args.no_peaks else None
    if args.veto_sigma > 0:   # the veto of PAPER.md:496-502 (the command of profiles/r03_refine_thread_ncu.md)
        from paper_2411_18370_b200 import binding as B
        p_hit = float(np.exp(-wl.rho_th)); w64 = np.asarray(wl.w, dtype=np.float64)
        r.ctx.set_option_f64(B.FT_OPT_WCOUNT_FLOOR, p_hit * w64.sum() + args.veto_sigma * np.sqrt(p_hit * (1.0 - p_hit) * (w64 ** 2).sum()))
    if args.antenna:   # sky-dependent weights (Eq. 4-5): the row-weighted tile kernel
        r.ctx.set_antenna(*W.antenna_geometry(wl))
    base_step = r.full_arrays_step() if args.full_arrays else r.step

    def step(c=None):
        cands = base_step(c)
        if args.full_arrays:
            return cands
        if world > 1:  # KBs of records: all-gather + merge under the same total order
            cands = S.merge_candidates(S.all_gather_candidates(S.to_global(cands, idx_off), dev if on_dev else None), wl.k,
                                       by_count=(wl.stat == "hough"))
        return cands

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warm = max(args.warmup, 3)
    c0 = r.ctx.counters()
    sampler = ClockSampler(local); sampler.start()
    ms, k_ms, n_launch = r.timed(args.steps, warm, flush, barrier, step)
    clocks = sampler.stop()
    c1 = r.ctx.counters()
    tot = torch.tensor([float(ms.sum())], device=dev if on_dev else "cpu")
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.MAX)
    total_ms = float(tot.item())
    value = r.evals * world * args.steps / (total_ms * 1e-3)

    # end to end through the C ABI from HOST buffers: H2D of the spectrogram (+ per-bin weights),
    # ft_create, ft_eval, ft_topk_per_band, candidates back on the host
    e2e_ms = []
    cands = None
    for s in range(max(2, min(args.steps, 5)) + 1):
        barrier()
        t0 = time.perf_counter()
        Pd = torch.empty_like(r.P_dev); Pd.copy_(r.P_host, non_blocking=True)
        wa = wl.w
        if wl.per_bin_weights:
            wa = torch.empty_like(r.w_arg); wa.copy_(r.w_host, non_blocking=True)
        c2 = r.make_ctx(Pd, wa)
        cands = step(c2)
        barrier()
        if s > 0:
            e2e_ms.append(1e3 * (time.perf_counter() - t0))
        c2.close()
    e2e_t = torch.tensor([float(np.mean(e2e_ms))], device=dev if on_dev else "cpu")
    if world > 1:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    h2d = r.P_host.numel() * 4 * (2 if wl.per_bin_weights else 1) + wl.n_sft * (8 + 24 + 4) + g.sky.size * 8
    d2h = int(cands.nbytes)

    if rank == 0:
        sm_mhz = clocks.get("sm_mhz") or 1965.0
        traffic_kernel = "ft_tile_kernel"
        if args.full_arrays and r.stat == "both" and args.config == 3:
            traffic_kernel = "ft_tileb_kernel"
        if args.full_arrays and r.stat == "hough" and args.config == 2:
            traffic_kernel = "ft_tile8_kernel"
        if args.antenna:
            traffic_kernel = "ft_tilew_kernel"
        traffic = args.traffic if args.traffic is not None else ncu_traffic(args.config, traffic_kernel)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warm, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": workload_config(wl, args, world, args.config),   # (the same dict on both arms)
            "step": {"statistic": r.stat,
                     "calls": "ft_eval, full arrays written out" if args.full_arrays else "ft_eval (bind) + ft_topk_per_band (fused selection)"},
            "templates_per_sec": value / wl.n_sft,
            "gpu_launches": int(c1["kernel_launches"] - c0["kernel_launches"]),
            "clocks": clocks,
            "e2e": {"value": r.evals * world / (float(e2e_t.item()) * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": d2h},
            "roofline": roofline_block(r.evals, k_ms, n_launch, total_ms / args.steps, peaks, measured, sm_mhz, traffic,
                                       "ft_tile_kernel (K2) / ft_generic_kernel (K0): the statistic launches of ft_topk_per_band, CUDA events on the library's stream around each launch, summed per step, mean over timed steps"),
            "measured_peaks": measured,
            "counters": {k: c1[k] for k in ("near_ties", "appended", "refined", "refine_fallbacks")},
            "kernel_geometry": r.ctx.describe(),
        }
        if world == 1 and not args.no_extra and args.config == 2 and not args.n_sky and not args.n_sft and not args.stat and not args.full_arrays and not args.antenna and not args.veto_sigma:
            out["extra"] = extra_runs(args, dev, flush, measured, peaks, None)
        if not args.no_cpu_baseline and world == 1:
            out["cpu_baseline"], _ = oracle_sample(wl, seconds=args.cpu_seconds)
        # the figures north_star's target names (all-sky, binary; plus per-bin weights), LAST in the line so that a
        # record that keeps only its tail still holds them: evals/s and fraction of the binding (shared-memory) roofline
        tg = {f"cfg{args.config}": {"value": value, "frac": out["roofline"]["frac"]}}
        for tag, key in (("cfg3", "cfg3_power_topk"), ("cfg3_both", "cfg3_both_topk"), ("cfg4", "cfg4_power_topk")):
            e = out.get("extra", {}).get(key)
            if e:
                tg[tag] = {"value": e["value"], "frac": e["roofline_frac"]}
        out["targets"] = tg
        print(json.dumps(out))
    r.close()
    if world > 1:
        dist.destroy_process_group()


def launcher_command(n: int, argv, port: int):
    """The command that starts n ranks of this script on this node (one per GPU; gloo: all on the visible GPU)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--n-sky", type=int, default=0)
    ap.add_argument("--n-sft", type=int, default=0)
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 generic, 2 tile")
    ap.add_argument("--fused", type=int, default=1)
    ap.add_argument("--tiles", type=int, default=0, help="f0 tiles (0 = library default)")
    ap.add_argument("--ppc", type=int, default=0, help="outer points per CTA (0 = library default)")
    ap.add_argument("--traffic", type=float, default=None, help="ncu dram bytes per launch (default: profiles/r02_dram_traffic.csv)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="gloo: exercise the N>1 path with every rank on one GPU (testing only)")
    ap.add_argument("--stat", default="", choices=["", "power", "hough", "both", "whough"], help="statistic (default: the configuration's)")
    ap.add_argument("--full-arrays", action="store_true", help="step = ft_eval with full statistic arrays written out, no selection")
    ap.add_argument("--only-bank", default="", choices=["", "isolated", "binary"],
                    help="run K1 alone: a xi-uniform random bank on the configuration's spectrogram")
    ap.add_argument("--antenna", action="store_true", help="sky-dependent weights w_a(n) (ft_set_antenna with the workload's detector geometry)")
    ap.add_argument("--veto-sigma", type=float, default=0.0,
                    help="> 0: power top-k under the weighted number-count floor mu + X sigma (PAPER.md:496-502); implies --stat both")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="headline configuration only")
    ap.add_argument("--no-peaks", action="store_true", help="skip ft_measure_peaks (roofline against nominal peaks)")
    ap.add_argument("--cpu-seconds", type=float, default=None)
    ap.add_argument("--bank", type=int, default=2_000_000, help="templates of the K1 random bank in `extra`")
    ap.add_argument("--sweep-max-templates", type=float, default=1.2e9)
    ap.add_argument("--sweep-min-templates", type=float, default=0.0)
    ap.add_argument("--sweep-reps", type=int, default=2)
    args = ap.parse_args(argv)
    args.cpu_seconds_set = args.cpu_seconds is not None
    if args.cpu_seconds is None:
        args.cpu_seconds = 15.0
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # start the ranks ourselves (the driver's own torchrun launch sets WORLD_SIZE and never comes here)
        sys.exit(subprocess.call(launcher_command(args.gpus, argv, _free_port())))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
