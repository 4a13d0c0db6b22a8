"""-m gpu: unstructured banks (ft_eval_templates, kernel K1) against the oracle's explicit-list
evaluation, element by element: counts bit-exact and power to 1e-5 outside flagged near-ties
(K1 evaluates the canonical fp64 arithmetic per evaluation, so power agrees to fp32 rounding)."""
import numpy as np
import pytest

from oracle import ft_oracle as fo
from paper_2411_18370_b200 import workloads as W

import ft_helpers as H

pytestmark = pytest.mark.gpu


def _run(ctx, tl, t_ref, stat="both", rho=1.6):
    import torch
    dev = torch.device("cuda:0")
    t = torch.from_numpy(tl.view(np.float64).reshape(-1, 8).copy()).to(dev)
    gp = torch.full((tl.size,), float("nan"), dtype=torch.float32, device=dev) if stat != "hough" else None
    gc = torch.full((tl.size,), -7, dtype=torch.int32, device=dev) if stat != "power" else None
    ctx.eval_templates(t, t_ref, stat, rho, gp, gc)
    return (gp.cpu().numpy() if gp is not None else None, gc.cpu().numpy() if gc is not None else None)


@pytest.mark.parametrize("cfg,n", [(2, 3001), (3, 2500), (4, 1777)])
def test_random_bank_matches_oracle(cfg, n):
    wl = {2: lambda: W.config2(n_sft=501, n_sky=7, band_hz=0.35),
          3: lambda: W.config3(n_sft=403, n_ap=3, n_porb=3, n_tasc=2, n_inj=0),
          4: lambda: W.config4(n_sft=300, n_sky=5, band_hz=0.4, n_lines=6)}[cfg]()
    tl = W.random_bank(wl, n, seed=1)
    o = fo.Oracle(wl)
    op, oc, _, otie = fo.eval_templates(o, tl.astype(fo.TEMPLATE_DTYPE), wl.grid.t_ref)
    ctx = H.gpu_context(wl)
    gp, gc = _run(ctx, tl, wl.grid.t_ref)
    ok = otie == 0
    assert np.array_equal(gc[ok], oc[ok])
    rel = np.abs(gp.astype(np.float64) - op) / op
    assert rel[ok].max() <= 1e-6, rel[ok].max()      # fp64 accumulation: only the final fp32 cast differs
    gp1, _ = _run(ctx, tl, wl.grid.t_ref, stat="power")
    _, gc1 = _run(ctx, tl, wl.grid.t_ref, stat="hough")
    assert np.array_equal(gp1, gp) and np.array_equal(gc1, gc)
    assert ctx.counters()["stat_launches"] == 1
    ctx.close()


def test_template_list_on_grid_equals_grid_evaluation_and_reference_time():
    """A list that enumerates config 1's grid gives ft_eval's arrays (same bins, same counts), also
    when f0 / f1 are referred to another t_ref (f1 = 0 there, so the values do not change)."""
    wl = H.apply_injections(W.config1())
    g = wl.grid
    ctx = H.gpu_context(wl)
    gp, gc = H.gpu_full(ctx, wl, stat="both")
    recs = [(g.f0_start + i * g.df0, 0.0, s[0], s[1], s[2], 0.0, 86400.0, 0.0) for s in g.sky for i in range(g.n_f0)]
    tl = np.array(recs, dtype=W.TEMPLATE_DTYPE)
    lp, lc = _run(ctx, tl, 12345.0)
    assert np.array_equal(lc, gc)
    assert np.allclose(lp, gp, rtol=2e-6, atol=0)
    ctx.close()


def test_out_of_range_track_is_an_error_not_a_clamp():
    from paper_2411_18370_b200 import binding as B
    wl = W.config1()
    tl = W.random_bank(wl, 64, seed=2)
    tl["f0"][5] += 1.0           # 1800 bins above the band
    ctx = H.gpu_context(wl)
    with pytest.raises(B.FtError) as e:
        _run(ctx, tl, 0.0)
    assert e.value.code == -4
    ctx.close()


def test_empty_list_is_ok():
    import torch
    wl = W.config1()
    ctx = H.gpu_context(wl)
    ctx.eval_templates(torch.empty(0, dtype=torch.float64, device="cuda:0"), 0.0, "power", 1.6, None, None)
    ctx.close()


# ---------------------------------------------------------------- arithmetic identities K1 relies on
def test_division_by_c_and_float_conversion_are_exact():
    """K1 divides v.n by c with a reciprocal multiply and one fused correction, and converts fp32 to fp64 with
    integer moves: both must equal the IEEE operations bit for bit (1e8 random quotients; every fp32 pattern)."""
    ctx = H.gpu_context(W.config1())
    assert ctx.selftest(0, 100_000_000, seed=3) == 0
    assert ctx.selftest(0, 10_000_000, seed=4) == 0
    assert ctx.selftest(1, 1 << 32) == 0
    assert ctx.selftest(2, 50_000_000, seed=5) == 0      # K1's orbital cosine against cos()
    ctx.close()


# ---------------------------------------------------------------- xi-uniform banks (Eq. A11), drawn on the device
def _box(wl, binary):
    g = wl.grid
    return dict(f0_lo=g.f0_start, f0_hi=g.f0_start + (g.n_f0 - 1) * g.df0, f1_lo=g.f1_start,
                f1_hi=g.f1_start + (g.n_f1 - 1) * g.df1, ra_lo=0.0, ra_hi=2 * np.pi, sd_lo=-1.0, sd_hi=1.0,
                ap_lo=float(np.min(g.a_p)) if binary else 0.0, ap_hi=float(np.max(g.a_p)) if binary else 0.0,
                porb_lo=float(np.min(g.P_orb)), porb_hi=float(np.max(g.P_orb)), t_ref=g.t_ref)


@pytest.mark.parametrize("cfg,binary", [(2, False), (3, True)])
def test_bank_draw_and_eval_bank_match_oracle(cfg, binary):
    """ft_bank_draw against the oracle's own implementation of the same counter-based xi-uniform draw (parameters to
    1e-13: pow / sin / cos differ in the last bits between the two libms), and ft_eval_bank (templates drawn in
    registers) against the oracle evaluating ITS bank: counts bit-exact, power to 1e-6 outside near-ties, and the
    loudest template of the batch."""
    import torch
    wl = {2: lambda: W.config2(n_sft=501, n_sky=7, band_hz=0.35),
          3: lambda: W.config3(n_sft=403, n_ap=3, n_porb=3, n_tasc=2, n_inj=0)}[cfg]()
    box = _box(wl, binary)
    if cfg == 3:   # fixed sky point of the binary config
        n = wl.grid.sky[0]
        ra = float(np.arctan2(n[1], n[0]) % (2 * np.pi))
        box.update(ra_lo=ra, ra_hi=ra, sd_lo=float(n[2]), sd_hi=float(n[2]))
    n, seed, first = 5000, 17, 123
    otl = fo.bank_draw(box, seed, first, n)
    ctx = H.gpu_context(wl)
    dev = torch.device("cuda:0")
    t = torch.zeros((n, 8), dtype=torch.float64, device=dev)
    ctx.bank_draw(box, seed, first, t)
    torch.cuda.synchronize()
    gtl = t.cpu().numpy().view(W.TEMPLATE_DTYPE).reshape(-1)
    for f in W.TEMPLATE_DTYPE.names:
        assert np.allclose(gtl[f], otl[f], rtol=1e-13, atol=1e-13 * (abs(box["t_ref"]) + 1)), f
    op, oc, owc, otie = fo.eval_templates(fo.Oracle(wl), otl, box["t_ref"])
    gp = torch.full((n,), float("nan"), dtype=torch.float32, device=dev)
    best, btp = ctx.eval_bank(box, seed, first, n, "power", wl.rho_th, out_power=gp)
    gp = gp.cpu().numpy()
    ok = otie == 0
    rel = np.abs(gp.astype(np.float64) - op) / op
    assert rel[ok].max() <= 1e-6
    assert int(otie.sum()) <= H.near_tie_bound(wl, n * wl.n_sft)
    j = int(np.lexsort((np.arange(n), -op))[0])
    if ok[j]:
        assert int(best["idx"]) == j
        assert abs(best["power"] - op[j]) <= 1e-12 * op[j] and best["count"] == oc[j]
        assert abs(best["wcount"] - owc[j]) <= 1e-12 * owc[j]
        assert abs(btp["f0"] - otl["f0"][j]) <= 1e-13 * otl["f0"][j]
    gc = torch.full((n,), -7, dtype=torch.int32, device=dev)
    bestc, _ = ctx.eval_bank(box, seed, first, n, "hough", wl.rho_th, out_count=gc)
    gc = gc.cpu().numpy()
    assert np.array_equal(gc[ok], oc[ok])
    jc = int(np.lexsort((np.arange(n), -oc))[0])
    assert int(bestc["idx"]) == jc or not ok[jc]
    ctx.close()


@pytest.mark.parametrize("cfg,binary", [(2, False), (3, True)])
def test_unstructured_bank_with_sky_dependent_weights(cfg, binary):
    """Eq. (4)-(5) on the path the paper uses them on (random banks): after ft_set_antenna,
    ft_eval_templates and ft_eval_bank weight every template by the antenna pattern of ITS sky point.  Against the
    oracle's explicit-list evaluation with the same antenna tables: power to 1e-6, counts bit-exact, the loudest
    template of a drawn batch; and the values differ from the fixed-weight ones (the feature is not vacuous)."""
    import torch
    wl = {2: lambda: W.config2(n_sft=501, n_sky=7, band_hz=0.35),
          3: lambda: W.config3(n_sft=403, n_ap=3, n_porb=3, n_tasc=2, n_inj=0)}[cfg]()
    ant = W.antenna_geometry(wl)
    o = fo.Oracle(wl, antenna=ant)
    ctx = H.gpu_context(wl)
    fixed_p, fixed_c = _run(ctx, W.random_bank(wl, 5003, seed=6), wl.grid.t_ref)
    ctx.set_antenna(*ant)
    for n in (5003, 700):           # with and without the f0 ordering
        tl = W.random_bank(wl, n, seed=6)
        if cfg == 3:                # several sky points, so that the weights differ between templates
            sky = W.config2(n_sft=8, n_sky=n).grid.sky
            tl["nx"], tl["ny"], tl["nz"] = sky[:, 0], sky[:, 1], sky[:, 2]
        op, oc, _, otie = fo.eval_templates(o, tl.astype(fo.TEMPLATE_DTYPE), wl.grid.t_ref)
        gp, gc = _run(ctx, tl, wl.grid.t_ref)
        ok = otie == 0
        assert np.array_equal(gc[ok], oc[ok])
        rel = np.abs(gp.astype(np.float64) - op) / op
        assert rel[ok].max() <= 1e-6, rel[ok].max()
        gp1, _ = _run(ctx, tl, wl.grid.t_ref, stat="power")
        assert np.array_equal(gp1, gp)
        if n == 5003 and cfg == 2:
            assert np.array_equal(gc, fixed_c) and np.abs(gp / fixed_p - 1).max() > 1e-3
    # a drawn bank: every statistic and the winner, which ft_eval_bank re-evaluates in fp64 with the same weights
    box = _box(wl, binary)
    n, seed, first = 4500, 23, 77
    otl = fo.bank_draw(box, seed, first, n)
    op, oc, owc, otie = fo.eval_templates(o, otl, box["t_ref"])
    dev = torch.device("cuda:0")
    gp = torch.full((n,), float("nan"), dtype=torch.float32, device=dev)
    best, _ = ctx.eval_bank(box, seed, first, n, "power", wl.rho_th, out_power=gp)
    gp = gp.cpu().numpy()
    ok = otie == 0
    assert (np.abs(gp.astype(np.float64) - op) / op)[ok].max() <= 1e-6
    j = int(np.lexsort((np.arange(n), -op))[0])
    if ok[j] and (np.sort(op)[-1] - np.sort(op)[-2]) > 1e-6 * op[j]:
        assert int(best["idx"]) == j
        assert abs(best["power"] - op[j]) <= 1e-12 * op[j] and best["count"] == oc[j]
        assert abs(best["wcount"] - owc[j]) <= 1e-12 * owc[j]
    # back to the weights as given
    ctx.set_antenna(None)
    back_p, back_c = _run(ctx, W.random_bank(wl, 5003, seed=6), wl.grid.t_ref)
    assert np.array_equal(back_p, fixed_p) and np.array_equal(back_c, fixed_c)
    ctx.close()


def test_track_of_a_template_equals_the_oracles():
    wl = W.config3(n_sft=403, n_ap=3, n_porb=3, n_tasc=2, n_inj=0)
    tl = W.random_bank(wl, 20, seed=5)
    o = fo.Oracle(wl)
    ctx = H.gpu_context(wl)
    for t in tl:
        k, x, rc = o.track_template(t, wl.grid.t_ref)
        assert rc == 0
        kg = ctx.track(t, wl.grid.t_ref)
        near = np.abs((x - np.floor(x)) - 0.5) < 1e-9
        assert np.array_equal(kg[~near], k[~near])
    ctx.close()


def test_mismatch_sampler_workload():
    """a signal injected along a template lambda in Gaussian noise; o N
    templates drawn uniformly in xi in a box around it; m = (s(lambda) - max s(lambda')) / (s(lambda) - mu_G)
    (Eq. 24).  The library's loudest template and its statistic equal the oracle's on the oracle's own bank, so
    the sampled mismatch is the same number; a denser bank gives a smaller mismatch."""
    import torch
    wl = W.config2(n_sft=400, n_sky=3, band_hz=0.2)
    g = wl.grid
    sig = np.zeros(1, dtype=W.TEMPLATE_DTYPE)
    n0 = g.sky[1]
    sig["f0"], sig["f1"] = g.f0_start + 0.1037, -3.3e-10
    sig["nx"], sig["ny"], sig["nz"] = n0
    sig["a_p"], sig["P_orb"], sig["t_asc"] = 0.0, 86400.0, 0.0
    o = fo.Oracle(wl)
    k, _, rc = o.track_template(sig[0], g.t_ref)
    assert rc == 0
    W.inject(wl.P, k, 3.0)                      # inputs: the oracle's track
    o = fo.Oracle(wl)
    s_sig = fo.eval_templates(o, sig, g.t_ref)[0][0]
    mu_G = float(wl.w.astype(np.float64).sum())
    ra0, sd0 = float(np.arctan2(n0[1], n0[0]) % (2 * np.pi)), float(n0[2])
    box = dict(f0_lo=float(sig["f0"][0]) - 3 * wl.df, f0_hi=float(sig["f0"][0]) + 3 * wl.df, f1_lo=-4e-10, f1_hi=-2.6e-10,
               ra_lo=ra0 - 0.02, ra_hi=ra0 + 0.02, sd_lo=max(-1.0, sd0 - 0.02), sd_hi=min(1.0, sd0 + 0.02),
               ap_lo=0.0, ap_hi=0.0, porb_lo=86400.0, porb_hi=86400.0, t_ref=g.t_ref)
    ctx = H.gpu_context(wl)
    ms = []
    for n in (300, 30000):
        otl = fo.bank_draw(box, 5, 0, n)
        op, _, _, otie = fo.eval_templates(o, otl, g.t_ref)
        j = int(np.lexsort((np.arange(n), -op))[0])
        m_oracle = float(fo.mismatch(s_sig, op[j], mu_G))
        best, _ = ctx.eval_bank(box, 5, 0, n, "power", wl.rho_th)
        m_gpu = (s_sig - best["power"]) / (s_sig - mu_G)
        if not otie[j]:
            assert int(best["idx"]) == j and abs(m_gpu - m_oracle) < 1e-12
        assert 0.0 <= m_gpu < 1.0
        ms.append(m_gpu)
    assert ms[1] <= ms[0]
    ctx.close()


def test_mismatch_sampler_against_the_oracles_sampler():
    """SURVEY §8(f) row 4 as a workload (paper_2411_18370_b200/sampler.py): N(Delta lambda) by
    Eq. (A10), o N templates per injected signal through ft_eval_bank, m by Eq. (24) -- against the oracle's own
    step-by-step sampler on the same streams: the same bank sizes, the same loudest template, s_best to fp64
    rounding, every m within 1e-5 (s(lambda) of the signal is the library's fp32 output); m < 1, and m is
    non-increasing in the oversampling for every signal (the banks of one stream are nested), hence its median
    (PAPER.md:326)."""
    from paper_2411_18370_b200 import sampler as S
    wl = W.config3(n_sft=403, n_ap=3, n_porb=3, n_tasc=2, n_inj=0)
    g = wl.grid
    n = g.sky[0]
    ra = float(np.arctan2(n[1], n[0]) % (2 * np.pi)); sd = float(n[2])
    f_mid = g.f0_start + 0.5 * g.n_f0 * g.df0
    box = dict(f0_lo=f_mid, f0_hi=f_mid + 0.01, f1_lo=0.0, f1_hi=0.0, ra_lo=ra, ra_hi=ra + 0.02, sd_lo=sd - 0.01, sd_hi=sd + 0.01,
               ap_lo=4.0, ap_hi=6.0, porb_lo=20 * 86400.0, porb_hi=25 * 86400.0, t_ref=g.t_ref)
    T_obs = float(wl.t_mid.max() - wl.t_mid.min()) + wl.T_sft
    N = S.n_templates(box, wl.T_sft, T_obs)
    assert abs(N - fo.n_templates(box, wl.T_sft, T_obs, 1e-4)) <= 1e-12 * N and 20 < N < 5000, N
    prev = None
    for o in (0.25, 2.0, 16.0):
        got = S.mismatch_samples(wl, box, n_inj=8, oversampling=o, seed=31, amp=3.0, T_obs=T_obs)
        ref = fo.mismatch_sampler(wl, box, 8, o, 31, 3.0, T_obs)
        assert got["n_bank"] == ref["n_bank"] == int(np.ceil(o * N)) and got["bank_templates"] == 8 * got["n_bank"]
        assert np.array_equal(got["best"], ref["best"])
        assert np.allclose(got["s_best"], ref["s_best"], rtol=1e-12, atol=0)
        assert np.allclose(got["s_signal"], ref["s_signal"], rtol=1e-6, atol=0)
        assert np.abs(got["m"] - ref["m"]).max() <= 1e-5
        assert np.all(got["m"] < 1.0) and np.all(got["m"] > -0.5)
        if prev is not None:
            assert np.all(got["m"] <= prev + 1e-12) and np.median(got["m"]) <= np.median(prev)
        prev = got["m"]
    assert np.median(prev) < 0.9      # sixteen-fold oversampling recovers a good part of the signal


@pytest.mark.parametrize("cfg,binary,antenna", [(2, False, False), (2, False, True), (3, True, True), (4, False, False)])
def test_loudest_of_a_random_bank_under_the_veto_by_z(cfg, binary, antenna):
    """ft_eval_bank_veto = the paper's per-box procedure on the unstructured path (Eq. 36):
    random bank, both statistics from one gather, weighted-count floor, loudest by z.  Against the oracle's
    eval_templates_z + loudest_of_bank on ITS draw of the same stream: the same winner (when no near-tie template
    and no fp64-rounding-level tie could change it), its refined power / wcount / z / sigma_G, and the full arrays."""
    import torch
    wl = {2: lambda: W.config2(n_sft=501, n_sky=7, band_hz=0.35),
          3: lambda: W.config3(n_sft=403, n_ap=3, n_porb=3, n_tasc=2, n_inj=0),
          4: lambda: W.config4(n_sft=300, n_sky=5, band_hz=0.4, n_lines=6)}[cfg]()
    ant = W.antenna_geometry(wl) if antenna else None
    o = fo.Oracle(wl, antenna=ant)
    box = _box(wl, binary)
    n, seed, first = 6000, 29, 11
    otl = fo.bank_draw(box, seed, first, n)
    op, oc, owc, otie, oz, osig = fo.eval_templates_z(o, otl, box["t_ref"])
    ctx = H.gpu_context(wl)
    if antenna:
        ctx.set_antenna(*ant)
    dev = torch.device("cuda:0")
    gp = torch.full((n,), float("nan"), dtype=torch.float32, device=dev)
    gc = torch.full((n,), -7, dtype=torch.int32, device=dev)
    floors = (0.0, float(np.quantile(owc, 0.9)), float(np.quantile(owc, 0.999)), 10.0 * float(owc.max()))
    for floor in floors:
        for by_z in (False, True):
            best, btp = ctx.eval_bank_veto(box, seed, first, n, wl.rho_th, floor, by_z, out_power=gp, out_count=gc)
            j = fo.loudest_of_bank(op, owc, oz, floor, by_z)
            if j < 0:
                assert best["idx"] == np.uint64(2 ** 64 - 1)
                continue
            key = oz if by_z else op
            passing = owc >= floor
            # unambiguous: the winner is clear of the runner-up and of the floor beyond fp64 rounding, no near-tie in reach
            runner = np.sort(key[passing])[-2] if passing.sum() > 1 else -np.inf
            clear = (key[j] - runner > 1e-9 * abs(key[j])) and not np.any((otie != 0) & (key >= key[j] - 0.2 * abs(key[j]))) \
                and np.min(np.abs(owc - floor)) > 1e-12
            if clear:
                assert int(best["idx"]) == j, (floor, by_z)
                tol = 1e-12 if antenna else 0.0
                assert abs(best["power"] - op[j]) <= tol * op[j] and best["count"] == oc[j]
                assert abs(best["wcount"] - owc[j]) <= max(tol, 1e-15) * owc[j]
                assert abs(best["z"] - oz[j]) <= 1e-9 * max(1.0, abs(oz[j])) and abs(best["sigma"] - osig[j]) <= 1e-12 * osig[j]
                assert abs(btp["f0"] - otl["f0"][j]) <= 1e-13 * otl["f0"][j]
    ok = otie == 0
    assert np.array_equal(gc.cpu().numpy()[ok], oc[ok])
    assert (np.abs(gp.cpu().numpy().astype(np.float64) - op) / op)[ok].max() <= 1e-6
    if antenna and cfg == 2:   # the order by z is not the order by power when sigma_G varies over the sky
        assert not np.array_equal(np.argsort(-oz)[:50], np.argsort(-op)[:50])
    ctx.close()
