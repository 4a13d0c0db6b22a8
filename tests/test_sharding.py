"""-m "not gpu": the N>1 path on CPU.  Two `gloo` ranks each take their shard of the bank
(paper_2411_18370_b200.sharding), select their per-band top-k (with the ORACLE standing in for the
GPU statistic: this test covers the host-side sharding / gather / merge logic, not the kernels),
all-gather the records and merge; rank 0 compares with the plain per-band sort of the whole bank."""
import os
import socket

import numpy as np
import pytest

from oracle import ft_oracle as fo
from paper_2411_18370_b200 import binding as B
from paper_2411_18370_b200 import sharding as S
from paper_2411_18370_b200 import workloads as W


def _cands_from_oracle(wl, k, bpb, by_count):
    o = fo.Oracle(wl)
    power, count, wcount, _ = o.eval_range()
    ref = fo.topk_per_band(count if by_count else power, wl.grid.n_f0, bpb, k)
    out = np.zeros((len(ref), k), dtype=B.CAND_DTYPE)
    out["idx"] = S.PAD
    for b, (idx, _) in enumerate(ref):
        j = idx.astype(np.int64)
        out["idx"][b, :len(j)] = idx
        out["power"][b, :len(j)] = power[j]
        out["wcount"][b, :len(j)] = wcount[j]
        out["count"][b, :len(j)] = count[j]
        out["band"][b] = b
    return out


def _make(cfg):
    if cfg == 2:
        return W.config2(n_sft=64, n_sky=5, band_hz=0.1)     # 5 sky points over 2 ranks: 2 + 3
    return W.config3(n_sft=48, n_ap=3, n_porb=2, n_tasc=2, n_inj=0)  # n_sky = 1: the a_p axis is sharded


def _worker(rank, world, port, cfg, by_count, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = _make(cfg)
        k, bpb = 4, int(round(wl.band_width / wl.grid.df0))
        n_bands = -(-wl.grid.n_f0 // bpb)
        g, off = S.shard_grid(wl.grid, rank, world)
        if g is None:
            local = np.zeros((n_bands, k), dtype=B.CAND_DTYPE)
            local["idx"] = S.PAD
        else:
            wl_local = W.Workload(wl.name, wl.config_id, wl.P, wl.t_mid, wl.vel, wl.w, wl.f_min, wl.df, g,
                                  wl.stat, wl.rho_th, wl.band_width, k, wl.T_sft)
            local = S.to_global(_cands_from_oracle(wl_local, k, bpb, by_count), off)
        merged = S.merge_candidates(S.all_gather_candidates(local), k, by_count)
        if rank == 0:
            ref = _cands_from_oracle(wl, k, bpb, by_count)
            q.put((np.array_equal(merged["idx"], ref["idx"]), np.array_equal(merged["power"], ref["power"]),
                   np.array_equal(merged["count"], ref["count"]), int(off)))
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("cfg,by_count,world", [(2, False, 2), (3, True, 2), (3, False, 2)])
def test_two_rank_shard_gather_merge_equals_global_topk(cfg, by_count, world):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, cfg, by_count, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[:3] == (True, True, True), res


def test_shard_grid_offsets_and_empty_shards():
    wl = _make(2)
    n_inner = wl.grid.n_f1 * wl.grid.n_f0
    seen = 0
    for r in range(3):
        g, off = S.shard_grid(wl.grid, r, 3)
        assert off == seen * n_inner
        seen += len(g.sky)
    assert seen == len(wl.grid.sky)
    one = W.Grid(f0_start=100.0, df0=1 / 1800, n_f0=8)  # every axis of length 1: rank 1 of 2 is empty
    assert S.shard_grid(one, 0, 2)[0] is None or S.shard_grid(one, 1, 2)[0] is None


def test_merge_orders_by_value_then_index_and_pads():
    a = np.zeros((1, 3), dtype=B.CAND_DTYPE); b = np.zeros((1, 3), dtype=B.CAND_DTYPE)
    a["idx"] = [[5, 9, S.PAD]]; a["power"] = [[2.0, 1.0, 0.0]]
    b["idx"] = [[7, 3, S.PAD]]; b["power"] = [[2.0, 1.0, 0.0]]
    m = S.merge_candidates([a, b], 3)
    assert m["idx"].tolist() == [[5, 7, 3]]           # ties in value broken by ascending index
    m5 = S.merge_candidates([a, b], 5)
    assert m5["idx"][0, 4] == S.PAD and m5["idx"][0, :4].tolist() == [5, 7, 3, 9]


def test_bench_starts_its_own_ranks():
    """`bench.py --gpus 2` without a launcher re-executes itself under torch.distributed.run (two ranks on
    127.0.0.1); here with the CPU reference arm so that no GPU is needed: rank 0 prints the one JSON line."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "1",
                        "--steps", "1", "--warmup", "0", "--cpu-seconds", "0.2"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["value"] > 0
    import bench
    cmd = bench.launcher_command(4, ["--gpus", "4", "--steps", "2"], 29999)
    assert cmd[1:6] == ["-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=4", "--master-addr"]
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and "127.0.0.1" in cmd
