"""The mismatch-distribution sampler of PAPER.md:320-324 as a workload of the library.

    For a parameter-space region Delta lambda, p(m | o) is sampled as follows:
      1. generate a Gaussian-noise data stream containing a CW signal according to the search's priors;
      2. uniformly sample o N(Delta lambda) templates in xi space and map them to lambda space;
      3. evaluate vmap s on the generated templates and compute m according to Eq. (24).

N(Delta lambda) is Eq. (29) with the density of Eq. (A9), i.e. the closed form of Eq. (A10); the
oversampling o is "the ratio of templates in the template bank over the number of templates in the covered region"
(:318).  Everything that touches the data runs in the library's kernels through the C ABI: the signal is template j
of a xi-uniform stream (ft_bank_draw), its track comes from ft_track, the bank is drawn and evaluated in registers
by ft_eval_bank (kernel K1), which also returns the loudest template re-evaluated in fp64.  This module only
orchestrates: it adds the signal to the caller's noise spectrogram (input preparation, on the device), loops over
injections and forms the scalar ratio of Eq. (24).  No CPU fallback; never imports oracle/."""
from __future__ import annotations

import math
import time

import numpy as np

from . import binding as B

BATCH = 1 << 24   # templates per ft_eval_bank call (the call takes n < 2^32; 16.8 M keeps the ordering scratch at 64 MiB)


def n_templates(box: dict, T_sft: float, T_obs: float, v_over_c: float = 1e-4) -> float:
    """N(Delta lambda) of Eq. (29) for the all-sky binary search: Eq. (A10), the integral of
    rho(lambda) = k f0^5 a_p^2 Omega^3 (Eq. A9), k = T_SFT^6 T_obs (v/c)^2, over the box (keys binding.BANK_FIELDS;
    sky as right ascension x sine of the declination, Omega = 2 pi / P_orb, phi_b over [0, 2 pi))."""
    if not box["ap_hi"] > 0.0:
        raise ValueError("n_templates: Eq. (A9)-(A10) are the binary search's; the box needs ap_hi > 0")
    k = (T_sft ** 6) * T_obs * (v_over_c ** 2)
    om = sorted((2.0 * math.pi / box["porb_lo"], 2.0 * math.pi / box["porb_hi"]))
    terms = ((box["f0_hi"] ** 6 - box["f0_lo"] ** 6) / 6.0,
             (box["ra_hi"] - box["ra_lo"]) * (box["sd_hi"] - box["sd_lo"]),
             (box["ap_hi"] ** 3 - box["ap_lo"] ** 3) / 3.0,
             (om[1] ** 4 - om[0] ** 4) / 4.0,
             2.0 * math.pi)
    return k * math.prod(terms)


def mismatch_samples(wl, box: dict, n_inj: int, oversampling: float, seed: int, amp: float, T_obs: float,
                     v_over_c: float = 1e-4, n_bank: int | None = None, device="cuda:0") -> dict:
    """n_inj samples of p(m | o) on the workload's noise spectrogram (per-SFT weights).

    Signal j = template j of the xi-uniform stream `seed` over `box`, added with amplitude `amp` to the spectrogram
    along its track; its bank = the first n_bank = ceil(o N) templates of stream `seed + 1 + j`.
    Returns m [n_inj] (Eq. 24 with mu_G = sum_a w_a), s_signal (fp32 statistic of the signal's own template),
    s_best (fp64, the loudest template of the bank), best (its position in the bank stream), n_bank, N, and the
    time spent drawing + evaluating banks (`bank_seconds`, host clock around the synchronising calls) with the
    templates that covers (`bank_templates`)."""
    import torch
    if wl.per_bin_weights:
        raise ValueError("mismatch_samples: per-SFT weights only (mu_G of Eq. 24 is sum_a w_a)")
    dev = torch.device(device)
    N = n_templates(box, wl.T_sft, T_obs, v_over_c)
    if n_bank is None:
        n_bank = max(1, int(math.ceil(oversampling * N)))
    mu_G = float(np.sum(np.asarray(wl.w, dtype=np.float64)))
    P0 = torch.from_numpy(np.ascontiguousarray(wl.P)).to(dev)
    rows = torch.arange(wl.n_sft, device=dev)
    ctx0 = B.Context(P0, wl.t_mid, wl.vel, wl.w, wl.f_min, wl.df)
    sig_dev = torch.zeros((1, 8), dtype=torch.float64, device=dev)
    sp = torch.zeros(1, dtype=torch.float32, device=dev)
    out = dict(m=np.empty(n_inj), s_signal=np.empty(n_inj), s_best=np.empty(n_inj), best=np.empty(n_inj, dtype=np.int64),
               n_bank=n_bank, N=N, bank_seconds=0.0, bank_templates=0)
    try:
        for j in range(n_inj):
            ctx0.bank_draw(box, seed, j, sig_dev)                         # step 1: a signal from the priors ...
            torch.cuda.synchronize(dev)
            sig = sig_dev.cpu().numpy().view(B.TEMPLATE_DTYPE).reshape(-1)[0]
            k = ctx0.track(sig, box["t_ref"])
            Pj = P0.clone()                                               # ... added to the noise along its track
            Pj[rows, torch.from_numpy(k).to(dev)] += amp
            ctx = B.Context(Pj, wl.t_mid, wl.vel, wl.w, wl.f_min, wl.df)
            try:
                ctx.eval_templates(sig_dev, box["t_ref"], "power", wl.rho_th, sp, None)
                s_sig = float(sp.item())
                best_v, best_i = -math.inf, -1
                t0 = time.perf_counter()
                for first in range(0, n_bank, BATCH):                     # steps 2-3: draw o N templates, vmap s, maximum
                    nb = min(BATCH, n_bank - first)
                    b, _ = ctx.eval_bank(box, seed + 1 + j, first, nb, "power", wl.rho_th)
                    if float(b["power"]) > best_v:                        # (ties: the lower index, i.e. the earlier batch)
                        best_v, best_i = float(b["power"]), first + int(b["idx"])
                out["bank_seconds"] += time.perf_counter() - t0
                out["bank_templates"] += n_bank
            finally:
                ctx.close()
            out["s_signal"][j], out["s_best"][j], out["best"][j] = s_sig, best_v, best_i
            out["m"][j] = (s_sig - best_v) / (s_sig - mu_G)               # Eq. (24)
    finally:
        ctx0.close()
    return out
