"""-m gpu: ft_eval_templates_noalloc, the handle-free entry point for hosts that must not allocate.

Some users of this library cannot let it call cudaMalloc: the process has given the whole GPU to one memory
pool (a raw allocation behind the pool's back fails, or breaks the pool's memory plan), or it runs a follow-up
loop with a latency budget (cudaMalloc / cudaFree stall every stream of the device), or its rule is simply "no
allocation after start-up".  For them the library keeps K1's work space -- the f0-ordered evaluation order,
its histogram, the out-of-range flag and the near-tie counter -- in a fixed array inside the library image, and
the caller passes every input and output itself.

What is checked here, through the C ABI: the entry point returns what the existing path (ft_create +
ft_eval_templates) returns, on two calls in a row -- the second with a different, shorter bank, so anything the
first call left in the shared array would show -- counts bit for bit and power within the 1e-5 relative tolerance
of the parity tests (the two paths run the same kernel, so the arrays are in fact identical); that the driver's
free-memory figure does not move across a call; and that a bank beyond the built-in maximum is refused with a
message instead of overrunning the array.

This file sorts last on purpose (pytest -x stops at the first failure): it must pass alone in a fresh process,
where its first call is also the device's set-up call, and after every other test."""
import numpy as np
import pytest

from paper_2411_18370_b200 import workloads as W

import ft_helpers as H

pytestmark = pytest.mark.gpu


def _device_inputs(wl):
    import torch
    dev = torch.device("cuda:0")
    return dict(P=torch.from_numpy(np.ascontiguousarray(wl.P)).to(dev),
                t_mid=torch.from_numpy(np.ascontiguousarray(wl.t_mid, dtype=np.float64)).to(dev),
                vel=torch.from_numpy(np.ascontiguousarray(wl.vel, dtype=np.float64)).to(dev),
                w=torch.from_numpy(np.ascontiguousarray(wl.w, dtype=np.float32)).to(dev))


def _existing_path(ctx, tl, t_ref, rho):
    import torch
    dev = torch.device("cuda:0")
    t = torch.from_numpy(tl.view(np.float64).reshape(-1, 8).copy()).to(dev)
    gp = torch.full((tl.size,), float("nan"), dtype=torch.float32, device=dev)
    gc = torch.full((tl.size,), -7, dtype=torch.int32, device=dev)
    ctx.eval_templates(t, t_ref, "both", rho, gp, gc)
    return gp.cpu().numpy(), gc.cpu().numpy()


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_noalloc_matches_existing_path_on_two_calls_in_a_row(cfg):
    """Isolated all-sky (per-SFT weights), binary (orbital cosine in the loop) and per-bin weights; each with a
    bank long enough for the f0 ordering in the static array (n >= 4096) followed by a shorter one."""
    import torch
    from paper_2411_18370_b200 import binding as B
    wl = {2: lambda: W.config2(n_sft=501, n_sky=7, band_hz=0.35),
          3: lambda: W.config3(n_sft=403, n_ap=3, n_porb=3, n_tasc=2, n_inj=0),
          4: lambda: W.config4(n_sft=300, n_sky=5, band_hz=0.4, n_lines=6)}[cfg]()
    dev = torch.device("cuda:0")
    d = _device_inputs(wl)
    ctx = H.gpu_context(wl)
    for call, (n, seed) in enumerate([(20011, 3), (6007, 4), (1500, 5)]):   # the last one: below the ordering threshold
        tl = W.random_bank(wl, n, seed=seed)
        want_p, want_c = _existing_path(ctx, tl, wl.grid.t_ref, wl.rho_th)
        t = torch.from_numpy(tl.view(np.float64).reshape(-1, 8).copy()).to(dev)
        gp = torch.full((n,), float("nan"), dtype=torch.float32, device=dev)
        gc = torch.full((n,), -7, dtype=torch.int32, device=dev)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info(dev)[0]
        ties = B.eval_templates_noalloc(d["P"], d["t_mid"], d["vel"], d["w"], wl.f_min, wl.df, t, wl.grid.t_ref, "both",
                                        wl.rho_th, gp, gc)
        free_after = torch.cuda.mem_get_info(dev)[0]
        got_p, got_c = gp.cpu().numpy(), gc.cpu().numpy()
        assert np.array_equal(got_c, want_c), (cfg, call)
        rel = np.abs(got_p.astype(np.float64) - want_p.astype(np.float64)) / np.abs(want_p.astype(np.float64))
        assert rel.max() <= H.POWER_RTOL, (cfg, call, rel.max())
        assert np.array_equal(got_p, want_p), (cfg, call)     # same kernel, same order of the sum
        assert 0 <= ties < 100
        if call > 0:   # (the very first call of a process may load the module: set-up, not steady state)
            assert free_after == free_before, (cfg, call, free_before - free_after)
    ctx.close()


def test_noalloc_single_statistics_and_size_limit():
    import torch
    from paper_2411_18370_b200 import binding as B
    wl = W.config2(n_sft=501, n_sky=7, band_hz=0.35)
    dev = torch.device("cuda:0")
    d = _device_inputs(wl)
    ctx = H.gpu_context(wl)
    tl = W.random_bank(wl, 5000, seed=9)
    want_p, want_c = _existing_path(ctx, tl, wl.grid.t_ref, wl.rho_th)
    t = torch.from_numpy(tl.view(np.float64).reshape(-1, 8).copy()).to(dev)
    gp = torch.empty(5000, dtype=torch.float32, device=dev)
    gc = torch.empty(5000, dtype=torch.int32, device=dev)
    B.eval_templates_noalloc(d["P"], d["t_mid"], d["vel"], d["w"], wl.f_min, wl.df, t, wl.grid.t_ref, "power", wl.rho_th, gp, None)
    B.eval_templates_noalloc(d["P"], d["t_mid"], d["vel"], d["w"], wl.f_min, wl.df, t, wl.grid.t_ref, "hough", wl.rho_th, None, gc)
    assert np.array_equal(gp.cpu().numpy(), want_p) and np.array_equal(gc.cpu().numpy(), want_c)
    # one template more than the built-in work space holds: refused up front, with a message, nothing launched
    too_many = torch.zeros((B.FT_NOALLOC_MAX_TEMPLATES + 1, 8), dtype=torch.float64, device=dev)
    with pytest.raises(B.FtError) as ei:
        B.eval_templates_noalloc(d["P"], d["t_mid"], d["vel"], d["w"], wl.f_min, wl.df, too_many, wl.grid.t_ref, "power",
                                 wl.rho_th, None, None)
    assert ei.value.code == -1 and "FT_NOALLOC_MAX_TEMPLATES" in str(ei.value)
    # a host pointer where device memory is expected is an argument error, not a fault
    lib = B.load_library()
    import ctypes as C
    msg = C.create_string_buffer(256)
    host_plain = np.zeros((16, 8))
    rc = lib.ft_eval_templates_noalloc(C.c_void_p(d["P"].data_ptr()), wl.n_sft, wl.n_bins, wl.n_bins,
                                       C.c_void_p(d["t_mid"].data_ptr()), C.c_void_p(d["vel"].data_ptr()),
                                       C.c_void_p(d["w"].data_ptr()), 1, wl.f_min, wl.df,
                                       host_plain.ctypes.data_as(C.c_void_p), 16, 0.0, 0, 1.6, None, None, None, None, msg, 256)
    assert rc == -1 and b"not device memory" in msg.value
    # a track outside the spectrogram: reported, that template NaN / -1, the others valid
    tl2 = tl[:4200].copy()
    tl2["f0"][7] = wl.f_min - 5.0
    t2 = torch.from_numpy(tl2.view(np.float64).reshape(-1, 8).copy()).to(dev)
    gp2 = torch.empty(4200, dtype=torch.float32, device=dev)
    gc2 = torch.empty(4200, dtype=torch.int32, device=dev)
    with pytest.raises(B.FtError) as ei:
        B.eval_templates_noalloc(d["P"], d["t_mid"], d["vel"], d["w"], wl.f_min, wl.df, t2, wl.grid.t_ref, "both", wl.rho_th, gp2, gc2)
    assert ei.value.code == -4
    p2, c2 = gp2.cpu().numpy(), gc2.cpu().numpy()
    assert np.isnan(p2[7]) and c2[7] == -1
    keep = np.arange(4200) != 7
    assert np.array_equal(p2[keep], want_p[:4200][keep]) and np.array_equal(c2[keep], want_c[:4200][keep])
    ctx.close()
