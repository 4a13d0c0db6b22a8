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
