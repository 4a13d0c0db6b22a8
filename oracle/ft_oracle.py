"""ctypes front-end of the CPU ORACLE (oracle/ft_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module; the product package never does, and nothing here imports the product's
CUDA binding.  It takes a `Workload`-like object (duck-typed: the seeded input module is the
only thing the two sides share) and returns numpy arrays.

The per-band top-k ("retrieving the loudest candidate within each region";
north_star: per-frequency-sub-band top-k) is the plain definition written out: sort every
template of a band by (ranking value descending, canonical index ascending), keep the first k.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import math

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libft_oracle.so")
_SRC = os.path.join(_HERE, "ft_oracle.c")


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (no FMA contraction: the canonical op order is literal)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
               "-std=c11", "-Wall", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


class _Problem(C.Structure):
    _fields_ = [
        ("P", C.c_void_p), ("n_sft", C.c_int64), ("n_bins", C.c_int64), ("ld", C.c_int64),
        ("t_mid", C.c_void_p), ("vel", C.c_void_p), ("w", C.c_void_p), ("wkind", C.c_int32),
        ("f_min", C.c_double), ("df", C.c_double),
        ("f0_start", C.c_double), ("df0", C.c_double), ("n_f0", C.c_int64),
        ("f1_start", C.c_double), ("df1", C.c_double), ("n_f1", C.c_int64),
        ("t_ref", C.c_double),
        ("n_sky", C.c_int64), ("sky", C.c_void_p),
        ("n_ap", C.c_int64), ("a_p", C.c_void_p),
        ("n_porb", C.c_int64), ("P_orb", C.c_void_p),
        ("n_tasc", C.c_int64), ("tasc_frac", C.c_void_p),
        ("rho_th", C.c_double),
        ("det_lat", C.c_void_p), ("det_gamma", C.c_void_p), ("lst", C.c_void_p),
    ]


class _BankBox(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("f0_lo", "f0_hi", "f1_lo", "f1_hi", "ra_lo", "ra_hi", "sd_lo", "sd_hi",
                                           "ap_lo", "ap_hi", "porb_lo", "porb_hi", "t_ref")]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.fto_track.restype = C.c_int
        _lib.fto_eval_range.restype = C.c_int
        _lib.fto_eval_list.restype = C.c_int
        _lib.fto_eval_templates.restype = C.c_int
        _lib.fto_num_threads.restype = C.c_int
        _lib.fto_eval_range_z.restype = C.c_int
        _lib.fto_track_template.restype = C.c_int
        _lib.fto_uniform.restype = C.c_double
        _lib.fto_uniform.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32]
        _lib.fto_antenna_ab.restype = None
        _lib.fto_antenna_ab.argtypes = [C.c_double] * 5 + [C.POINTER(C.c_double)] * 2
        _lib.fto_bank_draw.restype = None
    return _lib


def num_threads() -> int:
    return int(_load().fto_num_threads())


class Oracle:
    """Binds one workload (spectrogram + tables + grid) and evaluates templates on the CPU."""

    def __init__(self, wl, rho_th=None, antenna=None):
        """antenna: None (weights used as given) or (lat[n_sft], gamma[n_sft], lst[n_sft]) in radians:
        sky-dependent weights w_a(n) ∝ (a^2 + b^2) w_a normalised to sum 1 (Eq. 4-5)."""
        self.lib = _load()
        g = wl.grid
        self._keep = dict(
            P=np.ascontiguousarray(wl.P, dtype=np.float32),
            t_mid=np.ascontiguousarray(wl.t_mid, dtype=np.float64),
            vel=np.ascontiguousarray(wl.vel, dtype=np.float64),
            w=np.ascontiguousarray(wl.w, dtype=np.float32),
            sky=np.ascontiguousarray(g.sky, dtype=np.float64),
            a_p=np.ascontiguousarray(g.a_p, dtype=np.float64),
            P_orb=np.ascontiguousarray(g.P_orb, dtype=np.float64),
            tasc=np.ascontiguousarray(g.tasc_frac, dtype=np.float64),
        )
        if antenna is not None:
            for name, arr in zip(("det_lat", "det_gamma", "lst"), antenna):
                self._keep[name] = np.ascontiguousarray(arr, dtype=np.float64)
                assert self._keep[name].shape == (len(self._keep["t_mid"]),)
        k = self._keep
        n_sft, n_bins = k["P"].shape
        assert k["t_mid"].shape == (n_sft,) and k["vel"].shape == (n_sft, 3)
        wkind = 2 if k["w"].ndim == 2 else 1
        assert k["w"].shape == ((n_sft, n_bins) if wkind == 2 else (n_sft,))
        p = lambda a: a.ctypes.data_as(C.c_void_p)
        self.pb = _Problem(
            p(k["P"]), n_sft, n_bins, n_bins, p(k["t_mid"]), p(k["vel"]), p(k["w"]), wkind,
            float(wl.f_min), float(wl.df),
            float(g.f0_start), float(g.df0), int(g.n_f0),
            float(g.f1_start), float(g.df1), int(g.n_f1), float(g.t_ref),
            len(k["sky"]), p(k["sky"]), len(k["a_p"]), p(k["a_p"]),
            len(k["P_orb"]), p(k["P_orb"]), len(k["tasc"]), p(k["tasc"]),
            float(wl.rho_th if rho_th is None else rho_th),
            p(k["det_lat"]) if antenna is not None else None,
            p(k["det_gamma"]) if antenna is not None else None,
            p(k["lst"]) if antenna is not None else None)
        self.n_sft, self.n_bins = n_sft, n_bins
        self.dims = (len(k["sky"]), len(k["a_p"]), len(k["P_orb"]), len(k["tasc"]), int(g.n_f1),
                     int(g.n_f0))
        self.n_templates = int(np.prod([int(d) for d in self.dims], dtype=object))

    def track(self, idx: int):
        """bins k[n_sft] (int64), positions x[n_sft] (fp64) of one template; rc != 0 = out of range."""
        k = np.empty(self.n_sft, dtype=np.int64)
        x = np.empty(self.n_sft, dtype=np.float64)
        rc = self.lib.fto_track(C.byref(self.pb), C.c_uint64(int(idx)),
                                k.ctypes.data_as(C.c_void_p), x.ctypes.data_as(C.c_void_p))
        return k, x, rc

    def _outs(self, n):
        return (np.empty(n, np.float64), np.empty(n, np.int32), np.empty(n, np.float64),
                np.empty(n, np.uint8))

    def eval_range(self, begin: int = 0, end=None):
        """(power f64, count i32, wcount f64, near_tie u8) for canonical indices [begin, end)."""
        end = self.n_templates if end is None else end
        o = self._outs(end - begin)
        rc = self.lib.fto_eval_range(C.byref(self.pb), C.c_uint64(begin), C.c_uint64(end),
                                     *[a.ctypes.data_as(C.c_void_p) for a in o])
        if rc != 0:
            raise ValueError(f"oracle: a track left the spectrogram (rc={rc})")
        return o

    def eval_range_z(self, begin: int = 0, end=None):
        """(power, count, wcount, near_tie, z, sigma_G): eval_range plus the standardised statistic (Eq. 36)."""
        end = self.n_templates if end is None else end
        o = self._outs(end - begin) + (np.empty(end - begin, np.float64), np.empty(end - begin, np.float64))
        rc = self.lib.fto_eval_range_z(C.byref(self.pb), C.c_uint64(begin), C.c_uint64(end),
                                       *[a.ctypes.data_as(C.c_void_p) for a in o])
        if rc != 0:
            raise ValueError(f"oracle: a track left the spectrogram (rc={rc})")
        return o

    def track_template(self, template, t_ref: float):
        """bins and positions of one explicit template (a TEMPLATE_DTYPE record)."""
        tl = np.ascontiguousarray(np.atleast_1d(template), dtype=TEMPLATE_DTYPE)
        k = np.empty(self.n_sft, dtype=np.int64)
        x = np.empty(self.n_sft, dtype=np.float64)
        rc = self.lib.fto_track_template(C.byref(self.pb), tl.ctypes.data_as(C.c_void_p), C.c_double(float(t_ref)),
                                         k.ctypes.data_as(C.c_void_p), x.ctypes.data_as(C.c_void_p))
        return k, x, rc

    def eval_list(self, idx):
        idx = np.ascontiguousarray(idx, dtype=np.uint64)
        o = self._outs(idx.size)
        rc = self.lib.fto_eval_list(C.byref(self.pb), idx.ctypes.data_as(C.c_void_p),
                                    C.c_int64(idx.size), *[a.ctypes.data_as(C.c_void_p) for a in o])
        if rc != 0:
            raise ValueError(f"oracle: a track left the spectrogram (rc={rc})")
        return o


TEMPLATE_DTYPE = np.dtype([("f0", "<f8"), ("f1", "<f8"), ("nx", "<f8"), ("ny", "<f8"), ("nz", "<f8"),
                           ("a_p", "<f8"), ("P_orb", "<f8"), ("t_asc", "<f8")])


def eval_templates(oracle: "Oracle", templates, t_ref: float):
    """Unstructured bank: (power, count, wcount, near_tie) of an explicit
    list of templates (TEMPLATE_DTYPE records) on the oracle's spectrogram; grid axes unused."""
    tl = np.ascontiguousarray(templates, dtype=TEMPLATE_DTYPE)
    o = oracle._outs(tl.size)
    rc = oracle.lib.fto_eval_templates(C.byref(oracle.pb), tl.ctypes.data_as(C.c_void_p), C.c_int64(tl.size),
                                       C.c_double(float(t_ref)), *[a.ctypes.data_as(C.c_void_p) for a in o])
    if rc != 0:
        raise ValueError(f"oracle: a track left the spectrogram (rc={rc})")
    return o


def eval_templates_z(oracle: "Oracle", templates, t_ref: float):
    """eval_templates plus (z, sigma_G) of Eq. (36) for every template: (power, count, wcount, near_tie, z, sigma)."""
    tl = np.ascontiguousarray(templates, dtype=TEMPLATE_DTYPE)
    o = oracle._outs(tl.size) + (np.empty(tl.size, np.float64), np.empty(tl.size, np.float64))
    oracle.lib.fto_eval_templates_z.restype = C.c_int
    rc = oracle.lib.fto_eval_templates_z(C.byref(oracle.pb), tl.ctypes.data_as(C.c_void_p), C.c_int64(tl.size),
                                         C.c_double(float(t_ref)), *[a.ctypes.data_as(C.c_void_p) for a in o])
    if rc != 0:
        raise ValueError(f"oracle: a track left the spectrogram (rc={rc})")
    return o


def loudest_of_bank(power, wcount, z, wcount_floor: float = 0.0, rank_by_z: bool = False):
    """The paper's per-box step on a random bank (PAPER.md:476 "retrieve the loudest template per box", :496-502
    "loudest normalized power ... subject to a minimal weighted number count", Eq. 36 :346): among the templates
    whose weighted number count is >= wcount_floor, the one with the largest z (rank_by_z) or power; ties to the
    lower position.  Returns its position, or -1 if the veto leaves none."""
    key = np.asarray(z if rank_by_z else power, dtype=np.float64)
    keep = np.flatnonzero(np.asarray(wcount) >= wcount_floor)
    if keep.size == 0:
        return -1
    return int(keep[np.lexsort((keep, -key[keep]))[0]])


def topk_per_band(values, n_f0: int, bins_per_band: int, k: int, idx_begin: int = 0):
    """Plain definition of the per-band top-k over a FULL statistic array.

    values[j] is the ranking value of canonical index idx_begin + j (idx_begin a multiple of
    n_f0).  Band of a template = (idx % n_f0) // bins_per_band.  Returns a list over bands of
    (idx[k'], value[k']) sorted by (value desc, idx asc), k' = min(k, templates in band)."""
    values = np.asarray(values)
    idx = np.arange(values.size, dtype=np.uint64) + np.uint64(idx_begin)
    band = (idx % np.uint64(n_f0)).astype(np.int64) // bins_per_band
    n_bands = (n_f0 + bins_per_band - 1) // bins_per_band
    out = []
    for b in range(n_bands):
        sel = np.flatnonzero(band == b)
        order = np.lexsort((idx[sel], -values[sel].astype(np.float64)))[:k]
        out.append((idx[sel][order], values[sel][order]))
    return out


def topk_per_region(values, n_f0: int, bins_per_band: int, k: int, pbox=None, keep=None):
    """Plain definition of the per-region top-k over a FULL array (disjoint regions, the
    loudest candidates of each).  Region of canonical index idx = pbox[idx // n_f0] * n_bands +
    (idx % n_f0) // bins_per_band (pbox None: one box of points, i.e. frequency sub-bands).  keep: boolean
    mask of the templates that pass the number-count veto, None = all.  Returns a list
    over regions of (idx[k'], value[k']) sorted by (value desc, idx asc)."""
    values = np.asarray(values, dtype=np.float64)
    idx = np.arange(values.size, dtype=np.uint64)
    n_bands = (n_f0 + bins_per_band - 1) // bins_per_band
    band = (idx % np.uint64(n_f0)).astype(np.int64) // bins_per_band
    pt = (idx // np.uint64(n_f0)).astype(np.int64)
    pb = np.zeros(values.size, dtype=np.int64) if pbox is None else np.asarray(pbox, dtype=np.int64)[pt]
    region = pb * n_bands + band
    n_regions = (1 if pbox is None else int(np.max(pbox)) + 1) * n_bands
    ok = np.ones(values.size, dtype=bool) if keep is None else np.asarray(keep, dtype=bool)
    out = []
    for r in range(n_regions):
        sel = np.flatnonzero((region == r) & ok)
        order = np.lexsort((idx[sel], -values[sel]))[:k]
        out.append((idx[sel][order], values[sel][order]))
    return out


def mismatch(s_signal, s_template, mu_G):
    """Eq. (24): m(lambda'; lambda) = (s(lambda) - s(lambda')) / (s(lambda) - mu_G)."""
    return (np.asarray(s_signal, dtype=np.float64) - np.asarray(s_template, dtype=np.float64)) / \
        (np.asarray(s_signal, dtype=np.float64) - mu_G)


def n_templates(box: dict, T_sft: float, T_obs: float, v_over_c: float) -> float:
    """Eq. (29) for the all-sky binary search, i.e. Eq. (A10) PAPER.md:589-598 with the density of Eq. (A9)
    rho = k f0^5 a_p^2 Omega^3, k = T_SFT^6 T_obs (v/c)^2: the number of templates N(Delta lambda) that cover the
    lambda-box `box` (keys BANK_FIELDS; sky as (alpha, sin delta), Omega = 2 pi / P_orb, phi_b over its full range
    [0, 2 pi)).  Written out factor by factor in the order of Eq. (A10); f1 is not a resolved dimension there."""
    k = T_sft ** 6 * T_obs * v_over_c ** 2
    I_f0 = (box["f0_hi"] ** 6 - box["f0_lo"] ** 6) / 6.0                       # int df0 f0^5
    I_sky = (box["ra_hi"] - box["ra_lo"]) * (box["sd_hi"] - box["sd_lo"])      # int dalpha dsin(delta)
    I_ap = (box["ap_hi"] ** 3 - box["ap_lo"] ** 3) / 3.0                       # int da_p a_p^2
    Om_lo, Om_hi = 2.0 * math.pi / box["porb_hi"], 2.0 * math.pi / box["porb_lo"]
    I_Om = (Om_hi ** 4 - Om_lo ** 4) / 4.0                                     # int dOmega Omega^3
    I_phi = 2.0 * math.pi                                                      # int dphi_b
    return k * I_f0 * I_sky * I_ap * I_Om * I_phi


def mismatch_sampler(wl, box: dict, n_inj: int, oversampling: float, seed: int, amp: float, T_obs: float,
                     v_over_c: float = 1e-4, n_bank=None):
    """The sampling of p(m | o), step by step, for n_inj signals:
      1. a noise data stream (the workload's spectrogram) containing a CW signal drawn from the search's priors --
         signal j is template j of the xi-uniform stream `seed` over `box` (the density of Eq. A9), injected with
         amplitude `amp` along its own track (the bins of Eq. 2 at every SFT);
      2. o N(Delta lambda) templates (Eq. 29 / A10; rounded up, at least 1) drawn uniformly in xi over the box --
         the stream `seed + 1 + j`;
      3. the statistic of every one of them (Eq. 3) and m = (s(lambda) - max s(lambda')) / (s(lambda) - mu_G), Eq. (24),
         with mu_G = sum_a w_a (Eq. 13 on the P = s/2 scale).
    Returns dict(m [n_inj], s_signal, s_best, best [n_inj] positions in the bank stream, n_bank, N).  Per-SFT weights."""
    assert not wl.per_bin_weights
    N = n_templates(box, wl.T_sft, T_obs, v_over_c)
    if n_bank is None:
        n_bank = max(1, int(math.ceil(oversampling * N)))
    mu_G = float(np.sum(wl.w.astype(np.float64)))
    import copy
    m = np.empty(n_inj); s_sig = np.empty(n_inj); s_best = np.empty(n_inj); best = np.empty(n_inj, dtype=np.int64)
    for j in range(n_inj):
        sig = bank_draw(box, seed, j, 1)
        clean = Oracle(wl)
        k, _, rc = clean.track_template(sig[0], box["t_ref"])
        if rc != 0:
            raise ValueError("oracle: the signal's track leaves the spectrogram")
        wj = copy.copy(wl)
        wj.P = wl.P.copy()
        wj.P[np.arange(wl.n_sft), k] += np.float32(amp)
        oj = Oracle(wj)
        s_sig[j] = eval_templates(oj, sig, box["t_ref"])[0][0]
        bank = bank_draw(box, seed + 1 + j, 0, n_bank)
        sp = eval_templates(oj, bank, box["t_ref"])[0]
        best[j] = int(np.lexsort((np.arange(n_bank), -sp))[0])
        s_best[j] = sp[best[j]]
        m[j] = mismatch(s_sig[j], s_best[j], mu_G)
    return dict(m=m, s_signal=s_sig, s_best=s_best, best=best, n_bank=n_bank, N=N)


BANK_FIELDS = ("f0_lo", "f0_hi", "f1_lo", "f1_hi", "ra_lo", "ra_hi", "sd_lo", "sd_hi", "ap_lo", "ap_hi",
               "porb_lo", "porb_hi", "t_ref")


def bank_draw(box: dict, seed: int, first: int, n: int):
    """n templates drawn uniformly in the xi coordinates of Eq. (A11) over the lambda-box `box` (keys BANK_FIELDS),
    template i = first .. first + n - 1 of the counter-based stream `seed`."""
    lib = _load()
    bx = _BankBox(*[float(box[f]) for f in BANK_FIELDS])
    out = np.zeros(n, dtype=TEMPLATE_DTYPE)
    lib.fto_bank_draw(C.byref(bx), C.c_uint64(int(seed)), C.c_uint64(int(first)), C.c_int64(int(n)),
                      out.ctypes.data_as(C.c_void_p))
    return out


def uniform(seed: int, i: int, d: int) -> float:
    return float(_load().fto_uniform(int(seed), int(i), int(d)))


def antenna_ab(lat, gamma, lst, ra, dec):
    a, b = C.c_double(), C.c_double()
    _load().fto_antenna_ab(float(lat), float(gamma), float(lst), float(ra), float(dec), C.byref(a), C.byref(b))
    return a.value, b.value
