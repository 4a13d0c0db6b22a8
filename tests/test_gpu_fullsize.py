"""-m gpu: parity at BASELINE.json's FULL sizes (configs 2-4) in the launch configuration bench.py
times (auto kernel choice = tile kernel K2, fused top-k), on outputs the oracle can compute one by
one, plus properties that hold at any size; and the tile kernel's geometry edge cases (several f0
tiles, ragged tails, every points-per-CTA value class) at sizes the oracle finishes in seconds."""
import numpy as np
import pytest

from oracle import ft_oracle as fo
from paper_2411_18370_b200 import workloads as W

import ft_helpers as H

pytestmark = pytest.mark.gpu
PAD = np.uint64(2 ** 64 - 1)


def _full(cfg):
    return H.apply_injections({2: W.config2, 3: W.config3, 4: W.config4}[cfg]())


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_full_size_sampled_outputs_and_candidates(cfg):
    import torch
    wl = _full(cfg)
    g = wl.grid
    o = fo.Oracle(wl)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    ctx = H.gpu_context(wl)                       # kernel auto, fused top-k: what bench.py runs
    stat = "both" if wl.stat == "both" else "power"
    gp, gc = H.gpu_full(ctx, wl, stat=stat)
    assert "K2 tile kernel" in ctx.describe()
    # (a) sampled templates, one by one against the oracle (plus every injected template)
    rng = np.random.Generator(np.random.PCG64(100 + cfg))
    idx = rng.integers(0, g.n_templates, 4096).astype(np.uint64)
    inj = [int(g.ravel(*t)) for t, _ in wl.planned_injections]
    idx = np.unique(np.concatenate([idx, np.array(inj, dtype=np.uint64)]))
    op, oc, _, otie = o.eval_list(idx)
    j = idx.astype(np.int64)
    ok = otie == 0
    rel = np.abs(gp[j].astype(np.float64) - op) / op
    assert rel[ok].max() <= H.POWER_RTOL, f"max rel power error {rel[ok].max():.3e}"
    if gc is not None:
        assert np.array_equal(gc[j][ok], oc[ok])
    # (b) candidates: every one re-evaluated by the oracle, bit-identical value, total order
    ctx.eval(g, wl.stat, wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    assert cands.shape == (n_bands, wl.k) and np.all(cands["idx"] != PAD)
    flat = cands.reshape(-1)
    cp, cc, cw, _ = o.eval_list(flat["idx"])
    assert np.array_equal(flat["power"], cp) and np.array_equal(flat["count"], cc)
    assert np.array_equal(flat["wcount"], cw)
    for b in range(n_bands):
        c = cands[b]
        assert np.all((c["idx"] % np.uint64(g.n_f0)).astype(np.int64) // bpb == b)
        key = list(zip(-c["power"], c["idx"]))
        assert key == sorted(key), f"band {b} not in (value desc, idx asc) order"
    # (c) nothing louder was missed.  Whole bands against the ORACLE: every template of the band evaluated by the
    # oracle, its plain sort must give exactly the library's candidates, and the library's full fp32 array must
    # agree with it element by element (config 2: 9e6 templates x 4000 SFTs per band)
    for b in {2: (7,), 3: (0, 31), 4: (11,)}[cfg]:
        n_pt = g.n_templates // g.n_f0
        cols = np.arange(b * bpb, min(g.n_f0, (b + 1) * bpb), dtype=np.uint64)
        bidx = (np.arange(n_pt, dtype=np.uint64)[:, None] * np.uint64(g.n_f0) + cols[None, :]).reshape(-1)
        bp, bc, _, btie = o.eval_list(bidx)
        order = np.lexsort((bidx, -bp))[:wl.k]
        assert np.array_equal(cands[b]["idx"], bidx[order]), f"band {b}: candidates differ from the oracle's sort of the whole band"
        assert np.array_equal(cands[b]["power"], bp[order])
        okb = btie == 0
        relb = np.abs(gp[bidx.astype(np.int64)].astype(np.float64) - bp) / bp
        assert relb[okb].max() <= H.POWER_RTOL
        if gc is not None:
            assert np.array_equal(gc[bidx.astype(np.int64)][okb], bc[okb])
        assert int((~okb).sum()) <= H.near_tie_bound(wl, bidx.size * wl.n_sft)
    # ... and every other band against the library's own full array (a property, not parity: the fused
    # selection and the write-out agree)
    full = torch.from_numpy(gp).cuda().view(-1, g.n_f0)
    for b in range(n_bands):
        blk = full[:, b * bpb:(b + 1) * bpb]
        v, pos = torch.topk(blk.reshape(-1), wl.k)
        kth = float(cands[b]["power"][-1])
        w = blk.shape[1]
        tid = (pos // w) * g.n_f0 + b * bpb + (pos % w)
        must = tid[v.double() > kth * (1 + 2e-5)].cpu().numpy().astype(np.uint64)
        assert np.isin(must, cands[b]["idx"]).all(), f"band {b}: a louder template is missing"
        assert float(v[-1]) >= kth * (1 - 2e-5)
    # the loudest injected signal of a band is that band's rank-1 candidate (config 3: amplitudes
    # 0.5-3 against a noise maximum of ~1 + 5/sqrt(n_sft))
    loudest = {}
    for (t, amp) in wl.planned_injections:
        b = t[5] // bpb
        if b not in loudest or amp > loudest[b][1]:
            loudest[b] = (int(g.ravel(*t)), amp)
    for b, (tid, _) in loudest.items():
        assert int(cands[b, 0]["idx"]) == tid, f"band {b}: injection not at rank 1"
    ctx.close()


def test_config2_full_size_packed_number_count():
    """The packed number-count kernel (K2H, ft_tile8.cu) at the size bench.py times it at (config 2: 20 000 sky x
    1800 f0 x 5 f1 x 4000 SFTs, eighteen 224-SFT folds of the 8-bit lanes into the 16-bit level): the full count
    array against the oracle on 4096 sampled templates and on EVERY template of one sub-band, bit for bit; the
    top-10 by count of every band re-evaluated one by one, and that band's candidates against the oracle's sort."""
    wl = _full(2)
    g = wl.grid
    o = fo.Oracle(wl)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    ctx = H.gpu_context(wl)
    _, gc = H.gpu_full(ctx, wl, stat="hough")
    assert "packed tile kernel" in ctx.describe()
    rng = np.random.Generator(np.random.PCG64(212))
    idx = np.unique(rng.integers(0, g.n_templates, 4096).astype(np.uint64))
    _, oc, _, otie = o.eval_list(idx)
    ok = otie == 0
    assert np.array_equal(gc[idx.astype(np.int64)][ok], oc[ok])
    b = 13
    n_pt = g.n_templates // g.n_f0
    cols = np.arange(b * bpb, min(g.n_f0, (b + 1) * bpb), dtype=np.uint64)
    bidx = (np.arange(n_pt, dtype=np.uint64)[:, None] * np.uint64(g.n_f0) + cols[None, :]).reshape(-1)
    bp, bc, _, btie = o.eval_list(bidx)
    okb = btie == 0
    assert np.array_equal(gc[bidx.astype(np.int64)][okb], bc[okb])
    assert int((~okb).sum()) <= H.near_tie_bound(wl, bidx.size * wl.n_sft)
    ctx.eval(g, "hough", wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    assert cands.shape == (n_bands, wl.k) and np.all(cands["idx"] != PAD)
    flat = cands.reshape(-1)
    cp, cc, cw, _ = o.eval_list(flat["idx"])
    assert np.array_equal(flat["count"], cc) and np.array_equal(flat["power"], cp) and np.array_equal(flat["wcount"], cw)
    for bb in range(n_bands):
        c = cands[bb]
        assert np.all((c["idx"] % np.uint64(g.n_f0)).astype(np.int64) // bpb == bb)
        key = list(zip(-c["count"].astype(np.int64), c["idx"]))
        assert key == sorted(key)
    order = np.lexsort((bidx, -bc.astype(np.int64)))[:wl.k]
    # (a template flagged as a near-tie may legitimately differ by one hit: it matters only within one hit of the k-th count)
    risky = (~okb) & (bc >= bc[order[-1]] - 1)
    assert not risky.any(), "re-seed: a near-tie template sits at the selection boundary"
    assert np.array_equal(cands[b]["idx"], bidx[order]) and np.array_equal(cands[b]["count"], bc[order])
    ctx.close()


def test_config2_full_size_sky_dependent_weights():
    """The row-weighted tile kernel (K2W, ft_tilew.cu; Eq. 4-5) at the size bench.py times it at, with the paper's
    post-processing on top (loudest template per box of sky points x sub-band, ranked by z, Eq. 36): sampled
    outputs of the full array within 1e-5 of the oracle; every candidate re-evaluated by the oracle (the library
    evaluates a, b through per-SFT and per-sky tables: power, z, sigma_G to 1e-12, count exact); and one whole
    region (625 outer points x 90 f0 x 4000 SFTs) against the oracle's own sort of z."""
    wl = _full(2)
    g = wl.grid
    ant = W.antenna_geometry(wl)
    o = fo.Oracle(wl, antenna=ant)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    ctx = H.gpu_context(wl)
    ctx.set_antenna(*ant)
    gp, _ = H.gpu_full(ctx, wl, stat="power")
    assert "row-weighted" in ctx.describe()
    rng = np.random.Generator(np.random.PCG64(213))
    idx = np.unique(rng.integers(0, g.n_templates, 2048).astype(np.uint64))
    op, _, _, otie = o.eval_list(idx)
    ok = otie == 0
    rel = np.abs(gp[idx.astype(np.int64)].astype(np.float64) - op) / op
    assert rel[ok].max() <= H.POWER_RTOL, rel[ok].max()
    n_pt = g.n_templates // g.n_f0
    n_pbox = 160
    pbox = (np.arange(n_pt, dtype=np.int64) * n_pbox // n_pt).astype(np.int32)
    ctx.eval(g, "power", wl.rho_th)
    cands = ctx.topk_per_box(pbox, n_pbox, wl.band_width, 1, rank_by_z=True)
    assert cands.shape == (n_pbox * n_bands, 1) and np.all(cands["idx"] != PAD)
    flat = cands.reshape(-1)
    rsel = np.random.Generator(np.random.PCG64(214)).choice(flat.size, 400, replace=False)
    for c in flat[rsel]:
        i = int(c["idx"])
        p1, c1, w1, _, z1, s1 = o.eval_range_z(i, i + 1)
        assert abs(c["power"] - p1[0]) <= 1e-12 * p1[0] and c["count"] == c1[0]
        assert abs(c["z"] - z1[0]) <= 1e-9 * max(1.0, abs(z1[0])) and abs(c["sigma"] - s1[0]) <= 1e-12 * s1[0]
        assert c["box"] == pbox[i // g.n_f0] * n_bands + (i % g.n_f0) // bpb
    # one whole region: box 57 x band 6, every template by the oracle, plain sort of z
    pb, b = 57, 6
    pts = np.flatnonzero(pbox == pb)
    zs, ps, ids, tie = [], [], [], []
    for pt in pts:
        lo = int(pt) * g.n_f0 + b * bpb
        p1, _, _, t1, z1, _ = o.eval_range_z(lo, lo + bpb)
        zs.append(z1); ps.append(p1); ids.append(np.arange(lo, lo + bpb, dtype=np.uint64)); tie.append(t1)
    zs, ps, ids, tie = np.concatenate(zs), np.concatenate(ps), np.concatenate(ids), np.concatenate(tie)
    relr = np.abs(gp[ids.astype(np.int64)].astype(np.float64) - ps) / ps      # the full fp32 array on the whole region
    assert relr[tie == 0].max() <= H.POWER_RTOL
    j = int(np.lexsort((ids, -zs))[0])
    got = cands[pb * n_bands + b, 0]
    srt = np.sort(zs)
    # (a near-tie template may land one bin off: it matters only if its z is within reach of the top)
    assert not ((tie != 0) & (zs > srt[-1] - 1.0)).any() and srt[-1] - srt[-2] > 1e-9, "re-seed: ambiguous winner"
    assert int(got["idx"]) == int(ids[j]) and abs(got["z"] - zs[j]) <= 1e-9 * max(1.0, abs(zs[j]))
    ctx.close()


def test_config3_ranked_by_count_full_size():
    wl = _full(3)
    g = wl.grid
    o = fo.Oracle(wl)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    ctx = H.gpu_context(wl)
    ctx.eval(g, "hough", wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    flat = cands.reshape(-1)
    cp, cc, _, _ = o.eval_list(flat["idx"])
    assert np.array_equal(flat["count"], cc) and np.array_equal(flat["power"], cp)
    for b in range(n_bands):
        key = list(zip(-cands[b]["count"].astype(np.int64), cands[b]["idx"]))
        assert key == sorted(key)
    ctx.close()


GEOMETRY = [
    # (n_f0 via band_hz at T_SFT = 1800, n_sft, n_sky, points per CTA)
    (1.3, 77, 3, 0),     # 2340 f0 -> two f0 tiles, ragged last chunk, n_sft not a multiple of 4 or 32
    (1.3, 33, 4, 1),     # one point per CTA
    (0.35, 130, 9, 4),   # 630 f0, groups of 4 with a ragged last group (45 points)
    (0.02, 64, 2, 0),    # 36 f0: two chunks, second ragged
    (2.4, 40, 2, 3),     # 4320 f0: three tiles
]


@pytest.mark.parametrize("band_hz,n_sft,n_sky,ppc", GEOMETRY)
def test_tile_geometry_edge_cases(band_hz, n_sft, n_sky, ppc):
    wl = W.config2(n_sft=n_sft, n_sky=n_sky, band_hz=band_hz, band_width=0.01, k=3)
    o = fo.Oracle(wl)
    op, oc, _, otie = o.eval_range()
    ctx = H.gpu_context(wl, kernel=2, ppc=ppc)     # tile kernel forced: ineligible would raise
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    H.assert_full_parity(wl, gp, gc, op, oc, otie)
    bpb = int(round(wl.band_width / wl.grid.df0)); n_bands = -(-wl.grid.n_f0 // bpb)
    ctx.eval(wl.grid, "power", wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    H.assert_topk_parity(wl, cands, op, op, oc, wl.k, bpb)
    ctx.close()


TAILS = [
    # (n_f0, n_sft, n_sky, points per CTA, two points per warp expected)
    (450, 130, 5, 0, True),     # config 3's band: 14 x 32 + 2; 25 outer points: the last warp holds one point only
    (33, 77, 3, 0, True),       # 32 + 1
    (48, 64, 1, 0, True),       # 32 + 16: both tails fill the shared chunk; 5 points
    (49, 64, 2, 0, False),      # tail of 17: one point per warp
    (496, 40, 4, 2, True),      # 15 x 32 + 16, the widest; one warp (two points) per CTA
    (130, 203, 7, 5, True),     # 4 x 32 + 2; ppc = 5 -> two warps per CTA, ragged last group
    (64, 50, 2, 0, False),      # no tail at all
]


@pytest.mark.parametrize("n_f0,n_sft,n_sky,ppc,packed", TAILS)
def test_narrow_band_tail_packing(n_f0, n_sft, n_sky, ppc, packed):
    """Narrow bands of 32 m + t f0 (t <= 16) run two outer points per warp with the tails sharing one chunk
    (ft_tile2.cu): element-by-element parity with the oracle (power, count, candidates), and the same bits as the
    one-point-per-warp kernel (the accumulation order of a template does not change)."""
    from paper_2411_18370_b200 import binding as B
    wl = W.config2(n_sft=n_sft, n_sky=n_sky, band_hz=n_f0 / 1800.0, band_width=0.01 if n_f0 > 36 else n_f0 / 1800.0, k=3)
    assert wl.grid.n_f0 == n_f0
    o = fo.Oracle(wl)
    op, oc, _, otie = o.eval_range()
    ctx = H.gpu_context(wl, kernel=2, ppc=ppc)
    gp, _ = H.gpu_full(ctx, wl, stat="power", want_count=False)
    assert ("two points per warp" in ctx.describe()) == packed, ctx.describe()
    _, gc = H.gpu_full(ctx, wl, stat="hough")
    H.assert_full_parity(wl, gp, gc, op, oc, otie)
    bpb = int(round(wl.band_width / wl.grid.df0)); n_bands = -(-wl.grid.n_f0 // bpb)
    ctx.eval(wl.grid, "power", wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    H.assert_topk_parity(wl, cands, op, op, oc, wl.k, bpb)
    ctx.set_option(B.FT_OPT_TAIL_PACKING, 0)
    gp1, _ = H.gpu_full(ctx, wl, stat="power", want_count=False)
    assert "two points per warp" not in ctx.describe()
    assert np.array_equal(gp1, gp)
    ctx.close()


def test_generic_kernel_when_f0_step_differs_from_bin_width():
    """df0 = df/2 (a finer f0 grid than Eq. A1): not tileable, runs K0; forcing K2 is an error."""
    from paper_2411_18370_b200 import binding as B
    wl = W.config1()
    g = wl.grid
    fine = W.Grid(f0_start=g.f0_start, df0=g.df0 / 2, n_f0=2 * g.n_f0 - 1, sky=g.sky)
    wl2 = W.Workload("fine", 1, wl.P, wl.t_mid, wl.vel, wl.w, wl.f_min, wl.df, fine, "both", 1.6,
                     18 * fine.df0, 4, wl.T_sft)
    op, oc, _, otie = fo.Oracle(wl2).eval_range()
    ctx = H.gpu_context(wl2)
    gp, gc = H.gpu_full(ctx, wl2, stat="both")
    assert "K0" in ctx.describe()
    H.assert_full_parity(wl2, gp, gc, op, oc, otie)
    cands = ctx.topk_per_band(wl2.band_width, wl2.k, -(-fine.n_f0 // 18))
    H.assert_topk_parity(wl2, cands, op, op, oc, wl2.k, 18)
    ctx.set_option(B.FT_OPT_KERNEL, 2)
    with pytest.raises(B.FtError) as e:
        ctx.eval(fine, "power", 1.6)
    assert e.value.code == -7
    ctx.close()


@pytest.mark.parametrize("band_hz,n_sft,n_sky,ppc", [(1.3, 300, 3, 0), (2.4, 77, 2, 3), (0.6, 520, 5, 2)])
def test_packed_number_count_equals_fp32_map_and_oracle(band_hz, n_sft, n_sky, ppc):
    """The packed byte hit map (ft_tile8, 8-bit SIMD counters folded every 224 SFTs) and the fp32
    0/1 map give the same integer counts, equal to the oracle's; n_sft > 224 exercises the fold."""
    from paper_2411_18370_b200 import binding as B
    wl = W.config2(n_sft=n_sft, n_sky=n_sky, band_hz=band_hz, band_width=0.01, k=3)
    _, oc, _, otie = fo.Oracle(wl).eval_range()
    ctx = H.gpu_context(wl, kernel=2, ppc=ppc)
    _, gc8 = H.gpu_full(ctx, wl, stat="hough")
    assert "packed tile kernel" in ctx.describe()
    ctx.set_option(B.FT_OPT_PACKED_COUNT, 0)
    _, gc32 = H.gpu_full(ctx, wl, stat="hough")
    assert "packed" not in ctx.describe()
    assert np.array_equal(gc8, gc32)
    ok = otie == 0
    assert np.array_equal(gc8[ok], oc[ok])
    ctx.set_option(B.FT_OPT_PACKED_COUNT, 1)
    bpb = int(round(wl.band_width / wl.grid.df0)); n_bands = -(-wl.grid.n_f0 // bpb)
    ctx.eval(wl.grid, "hough", wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    op = fo.Oracle(wl).eval_range()[0]
    H.assert_topk_parity(wl, cands, oc, op, oc, wl.k, bpb, by_count=True)
    ctx.close()


def test_selection_overflow_recovery_and_forced_tiling():
    """The threshold sample is the first 296 CTA groups here (the bank is barely larger than the
    sample); 70 loud injections sit in the LAST a_p values, outside the sample, and flood the band's small append buffer (FT_OPT_SELECT_CAP) in the fused pass: the library tightens
    the threshold from the entries it kept and repeats the pass (refine_fallbacks > 0); the candidates
    still equal the oracle's.  Also forces 3 f0 tiles on a band one tile could hold."""
    from paper_2411_18370_b200 import binding as B
    wl = W.config3(n_sft=96, n_ap=24, n_porb=24, n_tasc=16, n_inj=0)
    rng = np.random.Generator(np.random.PCG64(11))
    wl.planned_injections = [((0, int(rng.integers(21, 24)), int(rng.integers(24)), int(rng.integers(16)), 0,
                               198 + int(rng.integers(9))), 3.0) for _ in range(70)]   # 70 loud tracks, one band (22)
    wl = H.apply_injections(wl)
    g = wl.grid
    o = fo.Oracle(wl)
    op, oc, _, _ = o.eval_range()
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    ctx = H.gpu_context(wl, kernel=2)
    ctx.set_option(B.FT_OPT_SELECT_CAP, 48)
    ctx.set_option(B.FT_OPT_F0_TILES, 3)
    ctx.eval(g, "power", wl.rho_th)
    assert "n_tiles=3" in ctx.describe()
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    H.assert_topk_parity(wl, cands, op, op, oc, wl.k, bpb)
    c = ctx.counters()
    assert c["refine_fallbacks"] >= 1, c
    ctx.close()


def test_config3_full_size_number_count_veto():
    """Config 3 at full size with the paper's floor (three sigma above the Gaussian-noise mean count,
    PAPER.md:502): every candidate re-evaluated by the oracle (count >= floor, power bit-identical,
    ordered), and nothing louder with a passing count was missed (masked top-k of the full arrays)."""
    import torch
    from paper_2411_18370_b200 import binding as B
    wl = _full(3)
    g = wl.grid
    o = fo.Oracle(wl)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    p_hit = float(np.exp(-wl.rho_th))
    floor = int(np.ceil(wl.n_sft * p_hit + 3.0 * np.sqrt(wl.n_sft * p_hit * (1 - p_hit))))
    ctx = H.gpu_context(wl)
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    ctx.set_option(B.FT_OPT_COUNT_FLOOR, floor)
    ctx.eval(g, "both", wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    live = cands["idx"] != PAD
    flat = cands[live]
    cp, cc, _, _ = o.eval_list(flat["idx"])
    assert np.array_equal(flat["power"], cp) and np.array_equal(flat["count"], cc) and np.all(cc >= floor)
    full = torch.from_numpy(np.where(gc >= floor, gp, -np.inf).astype(np.float32)).cuda().view(-1, g.n_f0)
    n_pass = 0
    for b in range(n_bands):
        c = cands[b][cands[b]["idx"] != PAD]
        key = list(zip(-c["power"], c["idx"]))
        assert key == sorted(key)
        blk = full[:, b * bpb:(b + 1) * bpb].reshape(-1)
        v, pos = torch.topk(blk, wl.k)
        n_ok = int(torch.isfinite(v).sum())
        assert len(c) == min(wl.k, int(torch.isfinite(blk).sum()))
        n_pass += len(c)
        if len(c):
            kth = float(c["power"][-1])
            w = bpb
            tid = (pos // w) * g.n_f0 + b * bpb + (pos % w)
            must = tid[:n_ok][v[:n_ok].double() > kth * (1 + 2e-5)].cpu().numpy().astype(np.uint64)
            assert np.isin(must, c["idx"]).all(), f"band {b}: a louder passing template is missing"
    assert n_pass > 0
    ctx.close()


@pytest.mark.parametrize("weighted", [True, False])
def test_veto_first_long_survivor_list_against_the_oracle(weighted):
    """Wide band (1 Hz at 200 Hz, config 2's spectrogram, 300 sky points = 2.7e6 templates) with a floor of mean +
    1 sigma: ~16 % of the bank survives the number-count pass (4e5 templates, evaluated for power one thread per
    candidate).  Oracle-exhaustive: the plain per-band sort of the masked full power array; refined values
    bit-identical; and the same candidates from the two bank-wide passes (FT_OPT_VETO_FIRST = 0)."""
    from paper_2411_18370_b200 import binding as B
    wl = W.config2(n_sky=300)
    g = wl.grid
    o = fo.Oracle(wl)
    op, oc, owc, _ = o.eval_range()
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    p_hit = float(np.exp(-wl.rho_th))
    w = wl.w.astype(np.float64)
    if weighted:
        floor = p_hit * w.sum() + 1.0 * np.sqrt(p_hit * (1 - p_hit) * (w ** 2).sum())
        keep = owc >= floor
    else:
        floor = int(np.ceil(wl.n_sft * p_hit + 1.0 * np.sqrt(wl.n_sft * p_hit * (1 - p_hit))))
        keep = oc >= floor
    assert 0.05 < keep.mean() < 0.3 and keep.sum() > 100_000
    ref = fo.topk_per_region(op, g.n_f0, bpb, wl.k, keep=keep)
    ctx = H.gpu_context(wl)
    if weighted:
        ctx.set_option_f64(B.FT_OPT_WCOUNT_FLOOR, floor)
    else:
        ctx.set_option(B.FT_OPT_COUNT_FLOOR, floor)
    got = {}
    for first in (1, 0):
        ctx.set_option(B.FT_OPT_VETO_FIRST, first)
        ctx.eval(g, "both", wl.rho_th)
        cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
        c = ctx.counters()
        assert (c["stat_launches"] == 1) == (first == 1), c
        if first:
            assert c["refined"] > 100_000      # the survivors, not a top-k superset
        H.assert_region_parity(cands, ref, op, {"power": op, "count": oc, "wcount": owc})
        got[first] = cands
    assert np.array_equal(got[0]["idx"], got[1]["idx"]) and np.array_equal(got[0]["power"], got[1]["power"])
    ctx.close()


def test_config2_full_size_weighted_count_veto_first():
    """Config 2 at full size under the paper's floor (weighted count three sigma above its Gaussian-noise mean,
    PAPER.md:502), in the launch configuration bench.py's `extra` times: the number-count pass alone, then its
    survivors (~2e5).  Every candidate re-evaluated by the oracle (bit-identical power / weighted count, floor
    respected, ordered), and the same candidates as the two bank-wide passes."""
    from paper_2411_18370_b200 import binding as B
    wl = _full(2)
    g = wl.grid
    o = fo.Oracle(wl)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    p_hit = float(np.exp(-wl.rho_th))
    w = wl.w.astype(np.float64)
    floor = p_hit * w.sum() + 3.0 * np.sqrt(p_hit * (1 - p_hit) * (w ** 2).sum())
    ctx = H.gpu_context(wl)
    ctx.set_option_f64(B.FT_OPT_WCOUNT_FLOOR, floor)
    got = {}
    for first in (1, 0):
        ctx.set_option(B.FT_OPT_VETO_FIRST, first)
        ctx.eval(g, "both", wl.rho_th)
        got[first] = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
        assert (ctx.counters()["stat_launches"] == 1) == (first == 1)
    assert np.array_equal(got[0]["idx"], got[1]["idx"]) and np.array_equal(got[0]["power"], got[1]["power"])
    cands = got[1]
    live = cands["idx"] != PAD
    assert live.sum() > 0
    flat = cands[live]
    cp, cc, cw, _ = o.eval_list(flat["idx"])
    assert np.array_equal(flat["power"], cp) and np.array_equal(flat["count"], cc) and np.array_equal(flat["wcount"], cw)
    assert np.all(cw >= floor)
    for b in range(n_bands):
        c = cands[b][cands[b]["idx"] != PAD]
        key = list(zip(-c["power"], c["idx"]))
        assert key == sorted(key) and np.all((c["idx"] % np.uint64(g.n_f0)) // np.uint64(bpb) == b)
    ctx.close()


def test_tight_orbit_limits_chunks_per_warp():
    """a_p Omega = 3.6e-3 (10 lt-s at P_orb = 0.2 d): the shift drifts by a bin every ~270 f0, so the plan
    must keep a warp's range short (32 J |D - 1| < 0.45) for the single-break model to hold; parity with
    the oracle element by element, several breaks per tile."""
    import math
    T_sft, n_sft, n_f0, pad = 900.0, 61, 700, 700
    df = 1.0 / T_sft
    rng = np.random.Generator(np.random.PCG64(321))
    t_mid = (np.arange(n_sft) * 7 + 0.5) * T_sft
    vel = W.earth_velocity(t_mid, *W.DETECTORS["H1"])
    n_bins = (n_f0 + 2 * pad + 3) // 4 * 4
    P = (-np.log(1.0 - rng.random((n_sft, n_bins)))).astype(np.float32)
    w = np.full(n_sft, 1.0 / n_sft, np.float32)
    ra, dec = 2.0, -0.3
    sky = np.array([[math.cos(dec) * math.cos(ra), math.cos(dec) * math.sin(ra), math.sin(dec)]])
    g = W.Grid(f0_start=150.0, df0=df, n_f0=n_f0, sky=sky, a_p=np.array([5.0, 10.0]),
               P_orb=np.array([0.2, 0.31]) * 86400.0, tasc_frac=np.array([0.0, 0.37, 0.8]))
    wl = W.Workload("tight-orbit", 7, P, t_mid, vel, w, 150.0 - pad * df, df, g, "both", 1.6, 70 * df, 4, T_sft)
    op, oc, _, otie = fo.Oracle(wl).eval_range()
    ctx = H.gpu_context(wl, kernel=2)
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    desc = ctx.describe()
    J = int(desc.split("J=")[1].split()[0])
    assert J <= 3, desc
    H.assert_full_parity(wl, gp, gc, op, oc, otie)
    cands = ctx.topk_per_band(wl.band_width, wl.k, 10)
    H.assert_topk_parity(wl, cands, op, op, oc, wl.k, 70)
    ctx.close()


@pytest.mark.parametrize("n_sft,n_sky,band_hz", [(1, 2, 0.05), (3, 1, 0.3), (5, 3, 0.02)])
def test_very_few_sfts(n_sft, n_sky, band_hz):
    """Degenerate time axis: fewer SFTs than one ring stage (4 rows) or one 32-SFT block."""
    wl = W.config2(n_sft=n_sft, n_sky=n_sky, band_hz=band_hz, band_width=0.01, k=2)
    op, oc, _, otie = fo.Oracle(wl).eval_range()
    ctx = H.gpu_context(wl, kernel=2)
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    H.assert_full_parity(wl, gp, gc, op, oc, otie)
    bpb = int(round(wl.band_width / wl.grid.df0)); n_bands = -(-wl.grid.n_f0 // bpb)
    ctx.eval(wl.grid, "power", wl.rho_th)
    cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
    H.assert_topk_parity(wl, cands, op, op, oc, wl.k, bpb)
    ctx.close()


# ---------------------------------------------------------------- BASELINE.json configs[4]: the scaling sweep
@pytest.mark.parametrize("size", [0, 1])
def test_config5_sweep_sizes_exhaustive(size):
    """Sweep sizes A1 (1e6 templates x 500 SFTs) and A2 (1e7 x 2000): every template against the oracle (full
    array, top-k fused and through the full write-out)."""
    from paper_2411_18370_b200 import binding as B
    n_sft, band_hz, n_sky = W.SWEEP_A[size]
    wl = W.config5(n_sft, band_hz, n_sky)
    g = wl.grid
    op, oc, _, otie = fo.Oracle(wl).eval_range()
    ctx = H.gpu_context(wl)
    gp, _ = H.gpu_full(ctx, wl, stat="power")
    assert "K2 tile kernel" in ctx.describe()
    flagged = H.assert_full_parity(wl, gp, None, op, oc, otie)
    assert flagged <= H.near_tie_bound(wl)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    for fused in (1, 0):
        ctx.set_option(B.FT_OPT_FUSED_TOPK, fused)
        ctx.eval(g, "power", wl.rho_th)
        cands = ctx.topk_per_band(wl.band_width, wl.k, n_bands)
        H.assert_topk_parity(wl, cands, op, op, oc, wl.k, bpb)
    ctx.close()


def test_config5_16000_sfts_and_4hz_band_geometry():
    """n_sft = 16 000 (the longest accumulation of the sweep: fp32 sums over the centred array must hold 1e-5) at a
    reduced sky grid, and the 4 Hz band of the largest sweep size, which plans several f0 tiles."""
    wl = W.config5(16000, 1.0, 8)
    op, oc, _, otie = fo.Oracle(wl).eval_range()
    ctx = H.gpu_context(wl)
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    H.assert_full_parity(wl, gp, gc, op, oc, otie)
    bpb = int(round(wl.band_width / wl.grid.df0)); n_bands = -(-wl.grid.n_f0 // bpb)
    ctx.eval(wl.grid, "power", wl.rho_th)
    H.assert_topk_parity(wl, ctx.topk_per_band(wl.band_width, wl.k, n_bands), op, op, oc, wl.k, bpb)
    ctx.close()
    wl = W.config5(64, 4.0, 6)
    op, oc, _, otie = fo.Oracle(wl).eval_range()
    ctx = H.gpu_context(wl)
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    desc = ctx.describe().split(";")[0]
    assert ("wpp=4" in desc and "n_tiles=2" in desc) or ("wpp=2" in desc and "n_tiles=4" in desc), desc   # several f0 tiles
    H.assert_full_parity(wl, gp, gc, op, oc, otie)
    bpb = int(round(wl.band_width / wl.grid.df0)); n_bands = -(-wl.grid.n_f0 // bpb)
    ctx.eval(wl.grid, "power", wl.rho_th)
    H.assert_topk_parity(wl, ctx.topk_per_band(wl.band_width, wl.k, n_bands), op, op, oc, wl.k, bpb)
    ctx.close()


def test_zero_velocity_straight_line_runs_the_tile_kernel():
    """v = 0, a_p = 0: D = 1 exactly, eps_bound = 0 (the J bound must not overflow).  The statistic
    is the weighted column sum of the spectrogram."""
    wl = W.config2(n_sft=200, n_sky=3, band_hz=0.5)
    wl.vel = np.zeros_like(wl.vel)
    wl.grid.n_f1, wl.grid.f1_start, wl.grid.df1 = 1, 0.0, 0.0
    ctx = H.gpu_context(wl, kernel=2)
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    assert "K2 tile kernel" in ctx.describe()
    k0 = int(round((wl.grid.f0_start - wl.f_min) / wl.df))
    col = (wl.w.astype(np.float64)[:, None] * wl.P.astype(np.float64)).sum(axis=0)[k0:k0 + wl.grid.n_f0]
    hits = (wl.P > np.float32(wl.rho_th)).sum(axis=0)[k0:k0 + wl.grid.n_f0]
    for i_sky in range(3):
        sl = slice(i_sky * wl.grid.n_f0, (i_sky + 1) * wl.grid.n_f0)
        assert np.allclose(gp[sl], col, rtol=1e-5) and np.array_equal(gc[sl], hits)
    ctx.close()


def test_config3_full_size_boxes_ranked_by_z():
    """Config 3 at full size, the paper's post-processing: 64 boxes of (a_p, P_orb, t_asc) points x 50 sub-bands,
    the loudest of each ranked by z (Eq. 36).  Every candidate re-evaluated by the oracle; the regions of two whole
    boxes of points against the oracle's exhaustive sort."""
    wl = _full(3)
    g = wl.grid
    o = fo.Oracle(wl)
    n_pt = g.n_templates // g.n_f0
    n_pbox = 64
    pbox = (np.arange(n_pt) * n_pbox // n_pt).astype(np.int32)
    bpb = int(round(wl.band_width / g.df0)); n_bands = -(-g.n_f0 // bpb)
    ctx = H.gpu_context(wl)
    ctx.eval(g, "both", wl.rho_th)
    cands = ctx.topk_per_box(pbox, n_pbox, wl.band_width, 1, rank_by_z=True)
    assert cands.shape == (n_pbox * n_bands, 1) and np.all(cands["idx"] != PAD)
    flat = cands.reshape(-1)
    cp, cc, cw, _ = o.eval_list(flat["idx"])
    assert np.array_equal(flat["power"], cp) and np.array_equal(flat["count"], cc) and np.array_equal(flat["wcount"], cw)
    w = wl.w.astype(np.float64)
    assert np.allclose(flat["z"], (cp - w.sum()) / np.sqrt((w ** 2).sum()), rtol=0, atol=1e-9)
    for pb in (0, 37):
        pts = np.flatnonzero(pbox == pb).astype(np.uint64)
        idx = (pts[:, None] * np.uint64(g.n_f0) + np.arange(g.n_f0, dtype=np.uint64)[None, :]).reshape(-1)
        bp = o.eval_list(idx)[0]
        band = (idx % np.uint64(g.n_f0)).astype(np.int64) // bpb
        for b in range(n_bands):
            m = band == b
            best = np.lexsort((idx[m], -bp[m]))[0]
            assert int(cands[pb * n_bands + b, 0]["idx"]) == int(idx[m][best]), (pb, b)
    ctx.close()


def test_bench_two_ranks_on_one_gpu_through_its_own_launcher():
    """`python bench.py --gpus 2 --dist-backend gloo`: bench.py starts both ranks itself; they share cuda:0, run
    independent shards (no kernel waits on another rank) and all-gather their candidates over gloo."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dist-backend", "gloo", "--n-sky", "600",
                        "--steps", "1", "--warmup", "3", "--no-peaks"], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["value"] > 0 and out["config"]["n_templates_per_gpu"] == 600 * 5 * 1800
