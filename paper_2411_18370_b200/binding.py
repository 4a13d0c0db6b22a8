"""Thin ctypes binding of libfasttracks_b200.so (include/fasttracks_b200.h): argument marshalling
only.  Every step of the path runs in the library's CUDA kernels; there is no CPU fallback and
this module never imports oracle/.  PyTorch supplies device memory and the stream."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

FT_STAT = {"power": 0, "hough": 1, "both": 2, "whough": 3}
FT_OPT_KERNEL, FT_OPT_FUSED_TOPK, FT_OPT_POINTS_PER_CTA, FT_OPT_PACKED_COUNT, FT_OPT_F0_TILES = 0, 1, 2, 3, 4
FT_OPT_SELECT_CAP, FT_OPT_COUNT_FLOOR, FT_OPT_ONE_PASS_BOTH, FT_OPT_WCOUNT_FLOOR, FT_OPT_VETO_FIRST, FT_OPT_TAIL_PACKING = 5, 6, 7, 8, 9, 10
SYMBOLS = ["ft_create", "ft_eval", "ft_topk_per_band", "ft_topk_per_box", "ft_set_antenna", "ft_eval_list",
           "ft_eval_templates", "ft_eval_templates_noalloc", "ft_bank_draw", "ft_eval_bank", "ft_eval_bank_veto", "ft_track", "ft_set_option", "ft_set_option_f64",
           "ft_get_counters", "ft_measure_peaks", "ft_selftest", "ft_last_error", "ft_describe", "ft_destroy"]


class FtGrid(C.Structure):
    _fields_ = [("f0_start", C.c_double), ("df0", C.c_double), ("n_f0", C.c_int64),
                ("f1_start", C.c_double), ("df1", C.c_double), ("n_f1", C.c_int32),
                ("t_ref", C.c_double),
                ("n_sky", C.c_int64), ("sky", C.c_void_p),
                ("n_ap", C.c_int32), ("a_p", C.c_void_p),
                ("n_porb", C.c_int32), ("P_orb", C.c_void_p),
                ("n_tasc", C.c_int32), ("tasc_frac", C.c_void_p)]


class FtCand(C.Structure):
    _fields_ = [("power", C.c_double), ("wcount", C.c_double), ("idx", C.c_uint64),
                ("count", C.c_int32), ("band", C.c_int32)]


CAND_DTYPE = np.dtype([("power", "<f8"), ("wcount", "<f8"), ("idx", "<u8"), ("count", "<i4"),
                       ("band", "<i4")])


CAND_BOX_DTYPE = np.dtype([("power", "<f8"), ("wcount", "<f8"), ("idx", "<u8"), ("count", "<i4"), ("box", "<i4"),
                           ("z", "<f8"), ("sigma", "<f8")])   # ft_cand_box

BANK_FIELDS = ("f0_lo", "f0_hi", "f1_lo", "f1_hi", "ra_lo", "ra_hi", "sd_lo", "sd_hi", "ap_lo", "ap_hi",
               "porb_lo", "porb_hi", "t_ref")


class FtBankBox(C.Structure):
    _fields_ = [(n, C.c_double) for n in BANK_FIELDS]


class FtPeaks(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("smem_gbs", "fp64_gflops", "fp64_cvt_gops", "l2_gbs", "sm_clock_mhz")]


TEMPLATE_DTYPE = np.dtype([("f0", "<f8"), ("f1", "<f8"), ("nx", "<f8"), ("ny", "<f8"), ("nz", "<f8"),
                           ("a_p", "<f8"), ("P_orb", "<f8"), ("t_asc", "<f8")])   # ft_template


class FtCounters(C.Structure):
    _fields_ = [("near_ties", C.c_uint64), ("refine_fallbacks", C.c_uint64),
                ("appended", C.c_uint64), ("refined", C.c_uint64),
                ("kernel_launches", C.c_uint64), ("stat_launches", C.c_uint64),
                ("last_kernel_ms", C.c_double)]


class FtError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"fasttracks_b200 error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path: str | None = None):
    """dlopen the in-tree shared library (fails loudly if it was not built)."""
    global _lib
    if _lib is None:
        if path is None:
            # in-tree library; compiled here with nvcc if it is missing or older than its sources
            # (raises if that fails: there is no fallback path)
            path = _build.build()
        if not os.path.exists(path):
            raise FileNotFoundError(f"{path} missing: run `python -m paper_2411_18370_b200.build`")
        lib = C.CDLL(path)
        lib.ft_create.restype = C.c_int
        lib.ft_create.argtypes = [C.POINTER(C.c_void_p), C.c_void_p, C.c_int64, C.c_int64, C.c_int64,
                                  C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_double,
                                  C.c_double, C.c_void_p]
        lib.ft_eval.restype = C.c_int
        lib.ft_eval.argtypes = [C.c_void_p, C.POINTER(FtGrid), C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        lib.ft_topk_per_band.restype = C.c_int
        lib.ft_topk_per_band.argtypes = [C.c_void_p, C.c_double, C.c_int32, C.c_void_p, C.POINTER(C.c_int32)]
        lib.ft_eval_list.restype = C.c_int
        lib.ft_eval_list.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        lib.ft_eval_templates.restype = C.c_int
        lib.ft_eval_templates.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_int, C.c_double,
                                          C.c_void_p, C.c_void_p]
        lib.ft_eval_templates_noalloc.restype = C.c_int
        lib.ft_eval_templates_noalloc.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p,
                                                  C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_int64,
                                                  C.c_double, C.c_int, C.c_double, C.c_void_p, C.c_void_p,
                                                  C.POINTER(C.c_uint64), C.c_void_p, C.c_char_p, C.c_int64]
        lib.ft_topk_per_box.restype = C.c_int
        lib.ft_topk_per_box.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_double, C.c_int32, C.c_int, C.c_void_p,
                                        C.POINTER(C.c_int32)]
        lib.ft_set_antenna.restype = C.c_int
        lib.ft_set_antenna.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.ft_bank_draw.restype = C.c_int
        lib.ft_bank_draw.argtypes = [C.c_void_p, C.POINTER(FtBankBox), C.c_uint64, C.c_uint64, C.c_int64, C.c_void_p]
        lib.ft_eval_bank.restype = C.c_int
        lib.ft_eval_bank.argtypes = [C.c_void_p, C.POINTER(FtBankBox), C.c_uint64, C.c_uint64, C.c_int64, C.c_int,
                                     C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.ft_eval_bank_veto.restype = C.c_int
        lib.ft_eval_bank_veto.argtypes = [C.c_void_p, C.POINTER(FtBankBox), C.c_uint64, C.c_uint64, C.c_int64, C.c_double,
                                          C.c_double, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.ft_track.restype = C.c_int
        lib.ft_track.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        lib.ft_set_option_f64.restype = C.c_int
        lib.ft_set_option_f64.argtypes = [C.c_void_p, C.c_int, C.c_double]
        lib.ft_measure_peaks.restype = C.c_int
        lib.ft_measure_peaks.argtypes = [C.c_void_p, C.POINTER(FtPeaks)]
        lib.ft_selftest.restype = C.c_int
        lib.ft_selftest.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.POINTER(C.c_uint64)]
        lib.ft_set_option.restype = C.c_int
        lib.ft_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int64]
        lib.ft_get_counters.restype = C.c_int
        lib.ft_get_counters.argtypes = [C.c_void_p, C.POINTER(FtCounters)]
        lib.ft_last_error.restype = C.c_char_p
        lib.ft_last_error.argtypes = [C.c_void_p]
        lib.ft_describe.restype = C.c_char_p
        lib.ft_describe.argtypes = [C.c_void_p]
        lib.ft_destroy.restype = None
        lib.ft_destroy.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


def _hp(a):
    return a.ctypes.data_as(C.c_void_p)


FT_NOALLOC_MAX_TEMPLATES = 1 << 20


def eval_templates_noalloc(P_dev, t_mid_dev, vel_dev, w_dev, f_min, df, templates_dev, t_ref, stat, rho_th,
                           out_power=None, out_count=None, n_bins=None, stream=None) -> int:
    """ft_eval_templates_noalloc: the statistic of an explicit template list without a handle and without any
    device allocation by the library -- for hosts whose device memory belongs to a pool, or that may not
    allocate after start-up (see the header).  Every array is a torch device tensor the CALLER allocated:
    P_dev fp32 [n_sft][ld], t_mid_dev fp64 [n_sft], vel_dev fp64 [n_sft][3], w_dev fp32 [n_sft] or [n_sft][ld],
    templates_dev n records of 64 B, out_power fp32 [n] / out_count int32 [n] or None.  At most
    FT_NOALLOC_MAX_TEMPLATES templates per call.  Marshalling only; returns the call's near-tie count."""
    import torch
    lib = load_library()
    assert P_dev.is_cuda and P_dev.dtype == torch.float32 and P_dev.dim() == 2 and P_dev.is_contiguous()
    n_sft, ld = P_dev.shape
    assert t_mid_dev.is_cuda and t_mid_dev.dtype == torch.float64 and t_mid_dev.numel() == n_sft and t_mid_dev.is_contiguous()
    assert vel_dev.is_cuda and vel_dev.dtype == torch.float64 and vel_dev.numel() == 3 * n_sft and vel_dev.is_contiguous()
    assert w_dev.is_cuda and w_dev.dtype == torch.float32 and w_dev.is_contiguous()
    assert w_dev.numel() in (n_sft, n_sft * ld)
    wkind = 1 if w_dev.dim() == 1 else 2
    assert templates_dev.is_cuda and templates_dev.is_contiguous()
    nbytes = templates_dev.numel() * templates_dev.element_size()
    assert nbytes % 64 == 0
    n = nbytes // 64
    for o in (out_power, out_count):
        assert o is None or (o.is_cuda and o.numel() == n and o.is_contiguous())
    pp = C.c_void_p(out_power.data_ptr()) if out_power is not None else None
    pc = C.c_void_p(out_count.data_ptr()) if out_count is not None else None
    st = stream if stream is not None else torch.cuda.current_stream(P_dev.device).cuda_stream
    ties = C.c_uint64(0)
    msg = C.create_string_buffer(512)
    with torch.cuda.device(P_dev.device):   # the call works on the current device
        rc = lib.ft_eval_templates_noalloc(C.c_void_p(P_dev.data_ptr()), n_sft, ld if n_bins is None else int(n_bins), ld,
                                           C.c_void_p(t_mid_dev.data_ptr()), C.c_void_p(vel_dev.data_ptr()),
                                           C.c_void_p(w_dev.data_ptr()), wkind, float(f_min), float(df),
                                           C.c_void_p(templates_dev.data_ptr()), n, float(t_ref), FT_STAT[stat],
                                           float(rho_th), pp, pc, C.byref(ties), C.c_void_p(st), msg, 512)
    if rc != 0:
        raise FtError(rc, msg.value.decode())
    return int(ties.value)


class Context:
    """ft_create / ft_eval / ft_topk_per_band on torch device tensors."""

    def __init__(self, P_dev, t_mid, vel, w, f_min, df, stream=None):
        import torch
        self.lib = load_library()
        self.h = C.c_void_p()
        assert P_dev.is_cuda and P_dev.dtype == torch.float32 and P_dev.dim() == 2 and P_dev.is_contiguous()
        n_sft, ld = P_dev.shape
        self.n_sft = n_sft
        t_mid = np.ascontiguousarray(t_mid, dtype=np.float64)
        vel = np.ascontiguousarray(vel, dtype=np.float64)
        if isinstance(w, torch.Tensor):  # per-(SFT, bin) weights live on the device
            assert w.is_cuda and w.dtype == torch.float32 and tuple(w.shape) == (n_sft, ld) and w.is_contiguous()
            wptr, wkind = C.c_void_p(w.data_ptr()), 2
        else:
            w = np.ascontiguousarray(w, dtype=np.float32)
            assert w.shape == (n_sft,)
            wptr, wkind = _hp(w), 1
        self._keep = (P_dev, w)
        self.stream = stream if stream is not None else torch.cuda.current_stream(P_dev.device)
        rc = self.lib.ft_create(C.byref(self.h), C.c_void_p(P_dev.data_ptr()), n_sft, ld, ld, _hp(t_mid),
                                _hp(vel), wptr, wkind, float(f_min), float(df),
                                C.c_void_p(self.stream.cuda_stream))
        self._check(rc)
        self.n_templates = 0
        self._n_f0, self._df0 = 1, 0.0

    def _check(self, rc):
        if rc != 0:
            msg = self.lib.ft_last_error(self.h).decode() if self.h else "no handle"
            raise FtError(rc, msg)

    def set_option(self, option: int, value: int):
        self._check(self.lib.ft_set_option(self.h, option, int(value)))

    def eval(self, grid, stat: str, rho_th: float, out_power=None, out_count=None):
        """grid: an object with the ft_grid fields (workloads.Grid).  out_*: torch device tensors or None."""
        ax = [np.ascontiguousarray(a, dtype=np.float64) for a in (grid.sky, grid.a_p, grid.P_orb, grid.tasc_frac)]
        g = FtGrid(float(grid.f0_start), float(grid.df0), int(grid.n_f0), float(grid.f1_start),
                   float(grid.df1), int(grid.n_f1), float(grid.t_ref), len(ax[0]), _hp(ax[0]),
                   len(ax[1]), _hp(ax[1]), len(ax[2]), _hp(ax[2]), len(ax[3]), _hp(ax[3]))
        self.n_templates = len(ax[0]) * len(ax[1]) * len(ax[2]) * len(ax[3]) * int(grid.n_f1) * int(grid.n_f0)
        self._n_f0, self._df0 = int(grid.n_f0), float(grid.df0)
        for o in (out_power, out_count):
            assert o is None or (o.is_cuda and o.numel() == self.n_templates and o.is_contiguous())
        pp = C.c_void_p(out_power.data_ptr()) if out_power is not None else None
        pc = C.c_void_p(out_count.data_ptr()) if out_count is not None else None
        self._check(self.lib.ft_eval(self.h, C.byref(g), FT_STAT[stat], float(rho_th), pp, pc))

    def topk_per_band(self, band_width_hz: float, k: int, n_bands_max: int = 0):
        # the C call writes n_bands * k records: size the buffer from the bound grid, not from the caller
        bpb = max(1, int(round(band_width_hz / self._df0))) if self._df0 > 0 else 1
        n_bands_max = max(int(n_bands_max), -(-self._n_f0 // bpb), 1)
        out = np.zeros((n_bands_max, k), dtype=CAND_DTYPE)
        nb = C.c_int32(0)
        self._check(self.lib.ft_topk_per_band(self.h, float(band_width_hz), int(k), _hp(out), C.byref(nb)))
        return out.reshape(-1)[: nb.value * k].reshape(nb.value, k)

    def set_option_f64(self, option: int, value: float):
        self._check(self.lib.ft_set_option_f64(self.h, option, float(value)))

    def set_antenna(self, lat=None, gamma=None, lst=None):
        """Per-SFT detector latitude, arm orientation and local sidereal angle (radians): sky-dependent weights."""
        if lat is None:
            self._check(self.lib.ft_set_antenna(self.h, None, None, None))
            return
        a = [np.ascontiguousarray(x, dtype=np.float64) for x in (lat, gamma, lst)]
        assert all(x.shape == (self.n_sft,) for x in a)
        self._check(self.lib.ft_set_antenna(self.h, _hp(a[0]), _hp(a[1]), _hp(a[2])))

    def topk_per_box(self, pbox, n_pbox: int, band_width_hz: float, k: int, rank_by_z: bool = False):
        """pbox: int32 [n_points] (or None).  Returns ft_cand_box records [n_regions][k]."""
        bpb = max(1, int(round(band_width_hz / self._df0))) if self._df0 > 0 else 1
        n_bands = max(-(-self._n_f0 // bpb), 1)
        n_pbox = int(n_pbox) if pbox is not None else 1
        out = np.zeros((n_pbox * n_bands, k), dtype=CAND_BOX_DTYPE)
        nr = C.c_int32(0)
        pb = None
        if pbox is not None:
            pb = np.ascontiguousarray(pbox, dtype=np.int32)
            assert pb.size * self._n_f0 == self.n_templates
        self._check(self.lib.ft_topk_per_box(self.h, _hp(pb) if pb is not None else None, n_pbox, float(band_width_hz),
                                             int(k), 1 if rank_by_z else 0, _hp(out), C.byref(nr)))
        return out.reshape(-1)[: nr.value * k].reshape(nr.value, k)

    @staticmethod
    def _box(box) -> "FtBankBox":
        return FtBankBox(*[float(box[f]) for f in BANK_FIELDS])

    def bank_draw(self, box: dict, seed: int, first: int, out_dev):
        """Fill a torch device tensor of n x 8 float64 with templates first .. first + n - 1 of a xi-uniform bank."""
        assert out_dev.is_cuda and out_dev.is_contiguous() and out_dev.numel() * out_dev.element_size() % 64 == 0
        n = out_dev.numel() * out_dev.element_size() // 64
        bx = self._box(box)
        self._check(self.lib.ft_bank_draw(self.h, C.byref(bx), int(seed), int(first), n, C.c_void_p(out_dev.data_ptr())))

    def eval_bank(self, box: dict, seed: int, first: int, n: int, stat: str, rho_th: float, out_power=None, out_count=None):
        """Draw + evaluate n templates of a xi-uniform bank; returns (best candidate record, best template record)."""
        for o in (out_power, out_count):
            assert o is None or (o.is_cuda and o.numel() == n and o.is_contiguous())
        pp = C.c_void_p(out_power.data_ptr()) if out_power is not None else None
        pc = C.c_void_p(out_count.data_ptr()) if out_count is not None else None
        best = np.zeros(1, dtype=CAND_DTYPE)
        tp = np.zeros(1, dtype=TEMPLATE_DTYPE)
        bx = self._box(box)
        self._check(self.lib.ft_eval_bank(self.h, C.byref(bx), int(seed), int(first), int(n), FT_STAT[stat], float(rho_th),
                                          pp, pc, _hp(best), _hp(tp)))
        return best[0], tp[0]

    def eval_bank_veto(self, box: dict, seed: int, first: int, n: int, rho_th: float, wcount_floor: float = 0.0,
                       rank_by_z: bool = False, out_power=None, out_count=None):
        """ft_eval_bank_veto: the loudest template (by z or power) among those passing the weighted-count floor;
        returns (ft_cand_box record, template record); record idx = 2^64 - 1 if none passes."""
        for o in (out_power, out_count):
            assert o is None or (o.is_cuda and o.numel() == n and o.is_contiguous())
        pp = C.c_void_p(out_power.data_ptr()) if out_power is not None else None
        pc = C.c_void_p(out_count.data_ptr()) if out_count is not None else None
        best = np.zeros(1, dtype=CAND_BOX_DTYPE)
        tp = np.zeros(1, dtype=TEMPLATE_DTYPE)
        bx = self._box(box)
        self._check(self.lib.ft_eval_bank_veto(self.h, C.byref(bx), int(seed), int(first), int(n), float(rho_th),
                                               float(wcount_floor), int(bool(rank_by_z)), pp, pc, _hp(best), _hp(tp)))
        return best[0], tp[0]

    def track(self, template, t_ref: float):
        tp = np.ascontiguousarray(np.atleast_1d(template), dtype=TEMPLATE_DTYPE)
        k = np.zeros(self.n_sft, dtype=np.int64)
        self._check(self.lib.ft_track(self.h, _hp(tp), float(t_ref), _hp(k)))
        return k

    def measure_peaks(self) -> dict:
        p = FtPeaks()
        self._check(self.lib.ft_measure_peaks(self.h, C.byref(p)))
        return {f: getattr(p, f) for f, _ in FtPeaks._fields_}

    def selftest(self, which: int, n: int, seed: int = 1) -> int:
        nf = C.c_uint64(0)
        self._check(self.lib.ft_selftest(self.h, int(which), int(n), int(seed), C.byref(nf)))
        return int(nf.value)

    def eval_list(self, idx):
        idx = np.ascontiguousarray(idx, dtype=np.uint64)
        out = np.zeros(idx.size, dtype=CAND_DTYPE)
        self._check(self.lib.ft_eval_list(self.h, _hp(idx), idx.size, _hp(out)))
        return out

    def eval_templates(self, templates_dev, t_ref: float, stat: str, rho_th: float, out_power=None, out_count=None):
        """templates_dev: torch uint8/float64 device tensor holding n ft_template records (64 B each)."""
        assert templates_dev.is_cuda and templates_dev.is_contiguous()
        nbytes = templates_dev.numel() * templates_dev.element_size()
        assert nbytes % 64 == 0
        n = nbytes // 64
        for o in (out_power, out_count):
            assert o is None or (o.is_cuda and o.numel() == n and o.is_contiguous())
        pp = C.c_void_p(out_power.data_ptr()) if out_power is not None else None
        pc = C.c_void_p(out_count.data_ptr()) if out_count is not None else None
        self._check(self.lib.ft_eval_templates(self.h, C.c_void_p(templates_dev.data_ptr()), n, float(t_ref),
                                               FT_STAT[stat], float(rho_th), pp, pc))

    def counters(self) -> dict:
        c = FtCounters()
        self._check(self.lib.ft_get_counters(self.h, C.byref(c)))
        return {f: getattr(c, f) for f, _ in FtCounters._fields_}

    def describe(self) -> str:
        return self.lib.ft_describe(self.h).decode()

    def close(self):
        if self.h:
            self.lib.ft_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
