"""Test-side glue: apply planned injections with the ORACLE's track, run the CUDA path through the
C-ABI binding, run the oracle, compare.  Lives in tests/ (the only place both sides may meet)."""
import numpy as np

from oracle import ft_oracle as fo
from paper_2411_18370_b200 import workloads as W

POWER_RTOL = 1e-5  # BASELINE.json north_star (4): normalized-power sums to 1e-5 relative


def apply_injections(wl):
    """Add each planned injection along the oracle's bins of that template (inputs only)."""
    if not wl.planned_injections:
        return wl
    o = fo.Oracle(wl)
    for idx_t, amp in wl.planned_injections:
        k, _, rc = o.track(int(wl.grid.ravel(*idx_t)))
        assert rc == 0
        W.inject(wl.P, k, amp)
    return wl


def gpu_context(wl, kernel=0, fused=1, ppc=0):
    import torch
    from paper_2411_18370_b200 import binding as B
    dev = torch.device("cuda:0")
    P = torch.from_numpy(np.ascontiguousarray(wl.P)).to(dev)
    w = torch.from_numpy(np.ascontiguousarray(wl.w)).to(dev) if wl.per_bin_weights else wl.w
    ctx = B.Context(P, wl.t_mid, wl.vel, w, wl.f_min, wl.df)
    ctx.set_option(B.FT_OPT_KERNEL, kernel)
    ctx.set_option(B.FT_OPT_FUSED_TOPK, fused)
    ctx.set_option(B.FT_OPT_POINTS_PER_CTA, ppc)
    return ctx


def gpu_full(ctx, wl, stat=None, rho_th=None, want_count=True):
    import torch
    stat = stat or wl.stat
    n = wl.grid.n_templates
    dev = torch.device("cuda:0")
    op = torch.full((n,), float("nan"), dtype=torch.float32, device=dev) if stat != "hough" else None
    oc = torch.full((n,), -1, dtype=torch.int32, device=dev) if (stat != "power" and want_count) else None
    ctx.eval(wl.grid, stat, wl.rho_th if rho_th is None else rho_th, op, oc)
    torch.cuda.synchronize()
    return (op.cpu().numpy() if op is not None else None, oc.cpu().numpy() if oc is not None else None)


def assert_full_parity(wl, gp, gc, o_power, o_count, o_tie):
    """Counts bit-exact and power within 1e-5 relative, except templates the oracle flags as
    within 1e-9 bin of a rounding tie (north_star (4)); returns the number flagged."""
    ok = o_tie == 0
    if gc is not None:
        bad = np.flatnonzero((gc != o_count) & ok)
        assert bad.size == 0, f"{bad.size} count mismatches, first idx {bad[:5]}: gpu {gc[bad[:5]]} oracle {o_count[bad[:5]]}"
    if gp is not None:
        rel = np.abs(gp.astype(np.float64) - o_power) / np.maximum(np.abs(o_power), 1e-300)
        bad = np.flatnonzero((rel > POWER_RTOL) & ok)
        assert bad.size == 0, f"{bad.size} power mismatches, max rel {rel[ok].max():.3e} at {bad[:5]}"
    return int((~ok).sum())


def assert_topk_parity(wl, cands, o_rank_values, o_power, o_count, k, bins_per_band, by_count=False):
    """Candidate SETS identical to the plain per-band sort of the oracle's full array, in order;
    refined fp64 power bit-identical to the oracle's, counts bit-exact."""
    ref = fo.topk_per_band(o_rank_values, wl.grid.n_f0, bins_per_band, k)
    assert cands.shape[0] == len(ref)
    for b, (ridx, _) in enumerate(ref):
        got = cands[b]
        n = len(ridx)
        assert np.array_equal(got["idx"][:n], ridx), f"band {b}: gpu {got['idx'][:n]} oracle {ridx}"
        assert np.all(got["idx"][n:] == np.uint64(2 ** 64 - 1))
        j = ridx.astype(np.int64)
        assert np.array_equal(got["power"][:n], o_power[j]), f"band {b}: refined power differs"
        assert np.array_equal(got["count"][:n], o_count[j])
        assert np.all(got["band"][:n] == b)


def near_tie_bound(wl, n_evals=None):
    """Flagged templates allowed: a few times the expected 2e-9 per evaluation (a tie window of 1e-9 bin on
    either side of x = k + 0.5, x uniform in the bin; SURVEY reading R17)."""
    n = wl.n_evals if n_evals is None else n_evals
    return max(3, int(10 * 2e-9 * n))


def assert_region_parity(cands, ref, value_of, exact_fields, tol_fields=(), rtol=1e-12):
    """cands[region][k] (binding.CAND_BOX_DTYPE / CAND_DTYPE) against the oracle's per-region plain sort `ref`
    (list of (idx, value)).  exact_fields: {field: oracle array} compared bit for bit; tol_fields likewise to rtol."""
    assert cands.shape[0] == len(ref), (cands.shape, len(ref))
    pad = np.uint64(2 ** 64 - 1)
    for r, (ridx, _) in enumerate(ref):
        got = cands[r]
        n = len(ridx)
        assert np.array_equal(got["idx"][:n], ridx), f"region {r}: gpu {got['idx'][:n]} oracle {ridx}"
        assert np.all(got["idx"][n:] == pad), f"region {r}: padding"
        j = ridx.astype(np.int64)
        for f, arr in exact_fields.items():
            assert np.array_equal(got[f][:n], arr[j]), f"region {r}: {f} differs"
        for f, arr in tol_fields:
            assert np.allclose(got[f][:n], arr[j], rtol=rtol, atol=1e-9 if f == "z" else 0), f"region {r}: {f} differs"
