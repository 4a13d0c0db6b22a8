"""Seeded synthetic inputs shaped like the paper's O3 workloads.

This module is the ONE thing the oracle (tests) and the CUDA path (tests, bench.py) share.
It holds NONE of the method's arithmetic: no track, no bin index, no statistic.  Where an
input needs a track (an injected signal, "data stream containing a CW signal"),
the caller hands in the bins; `inject()` only adds an amplitude at given (row, bin) pairs.

What it synthesises (stand-ins for LVK O3a open data, not in this box):
  * the normalized spectrogram P[alpha][k] ~ Exponential(1) (Eq. 11 chi^2_2 / 2,
    footnote 2 :141), fp32;
  * SFT mid-times with gaps (PAPER.md:74 footnote 1) from a duty-cycle mask;
  * detector velocity from an analytic circular-orbit + sidereal-rotation Earth model
    (BASELINE.json configs[0]);
  * weights w_alpha ∝ 1/S_alpha normalised to sum 1 (PAPER.md:69 Eq. 4, :84 Eq. 5), or per-bin
    weights with non-stationary lines (BASELINE.json configs[3]);
  * template-grid axes (f0, f1, sky, a_p, P_orb, t_asc fractions).

numpy's PCG64 bit stream and `Generator.random` (53-bit uniforms) are version-stable;
Exponential(1) is drawn as -log(u) so no library sampling algorithm is involved.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

BASE_SEED = 241118370
C_LIGHT = 299792458.0

# stream ids (one generator per array)
_S_P, _S_PSD, _S_DUTY, _S_SUB, _S_INJ, _S_LINES = 0, 1, 2, 3, 4, 5

# (latitude deg, longitude deg) — LHO, LLO as BASELINE.json configs[1] names them
DETECTORS = {"H1": (46.455, -119.408), "L1": (30.563, -90.774), "cfg1": (46.45, 0.0)}


def _rng(config_id: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64((BASE_SEED + config_id) * 16 + stream))


def _uniform_open(rng: np.random.Generator, shape) -> np.ndarray:
    """u in (0,1): never 0, so -log(u) is finite."""
    u = rng.random(shape)
    return np.where(u <= 0.0, 2.0 ** -54, u)


def exponential_spectrogram(rng: np.random.Generator, n_sft: int, n_bins: int) -> np.ndarray:
    out = np.empty((n_sft, n_bins), dtype=np.float32)
    step = max(1, (1 << 22) // max(n_bins, 1))
    for a in range(0, n_sft, step):
        b = min(n_sft, a + step)
        out[a:b] = (-np.log(_uniform_open(rng, (b - a, n_bins)))).astype(np.float32)
    return out


def earth_velocity(t: np.ndarray, lat_deg: float, lon_deg: float) -> np.ndarray:
    """Detector velocity, equatorial Cartesian, m/s: circular orbit 29.78 km/s tilted by
    23.44 deg plus 465 m/s * cos(lat) sidereal rotation (BASELINE.json configs[0])."""
    t = np.asarray(t, dtype=np.float64)
    v_o, eps = 29780.0, math.radians(23.44)
    phi_o = 2.0 * math.pi * t / (365.25636 * 86400.0)
    v_r = 465.0 * math.cos(math.radians(lat_deg))
    phi_r = 2.0 * math.pi * t / 86164.0905 + math.radians(lon_deg)
    v = np.empty((t.size, 3), dtype=np.float64)
    v[:, 0] = -v_o * np.sin(phi_o) - v_r * np.sin(phi_r)
    v[:, 1] = v_o * np.cos(phi_o) * math.cos(eps) + v_r * np.cos(phi_r)
    v[:, 2] = v_o * np.cos(phi_o) * math.sin(eps)
    return v


def fibonacci_sphere(n: int) -> np.ndarray:
    """Deterministic near-uniform sky grid: z_j = 1-(2j+1)/n, phi_j = 2 pi j / golden."""
    j = np.arange(n, dtype=np.float64)
    z = 1.0 - (2.0 * j + 1.0) / n
    phi = 2.0 * math.pi * j / ((1.0 + math.sqrt(5.0)) / 2.0)
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1)


def duty_cycle_slots(rng_mask, rng_sub, n_slots: int, n_keep: int, duty: float = 0.7,
                     mean_on: float = 16.0) -> np.ndarray:
    """On/off mask with exponential run lengths (mean on-run `mean_on` slots, duty cycle
    `duty`), then exactly n_keep on-slots drawn without replacement, sorted."""
    mean_off = mean_on * (1.0 - duty) / duty
    mask = np.zeros(n_slots, dtype=bool)
    pos, on = 0, True
    while pos < n_slots:
        run = 1 + int(-math.log(float(_uniform_open(rng_mask, ()))) * (mean_on if on else mean_off))
        if on:
            mask[pos:pos + run] = True
        pos += run
        on = not on
    on_slots = np.flatnonzero(mask)
    if on_slots.size < n_keep:  # tiny test sizes: fall back to every slot
        on_slots = np.arange(n_slots)
    pick = rng_sub.permutation(on_slots.size)[:n_keep]
    return np.sort(on_slots[pick])


@dataclass
class Grid:
    """Template grid, the axes of ft_grid (include/fasttracks_b200.h)."""
    f0_start: float
    df0: float
    n_f0: int
    f1_start: float = 0.0
    df1: float = 0.0
    n_f1: int = 1
    t_ref: float = 0.0
    sky: np.ndarray = field(default_factory=lambda: np.array([[0.0, 0.0, 1.0]]))
    a_p: np.ndarray = field(default_factory=lambda: np.zeros(1))
    P_orb: np.ndarray = field(default_factory=lambda: np.array([86400.0]))
    tasc_frac: np.ndarray = field(default_factory=lambda: np.zeros(1))

    @property
    def dims(self):
        """(n_sky, n_ap, n_porb, n_tasc, n_f1, n_f0), slowest to fastest."""
        return (len(self.sky), len(self.a_p), len(self.P_orb), len(self.tasc_frac),
                self.n_f1, self.n_f0)

    @property
    def n_templates(self) -> int:
        return int(np.prod([int(d) for d in self.dims], dtype=object))

    def unravel(self, idx):
        return np.unravel_index(np.asarray(idx, dtype=np.int64), self.dims)

    def ravel(self, i_sky, i_ap, i_porb, i_tasc, i_f1, i_f0):
        return np.ravel_multi_index((i_sky, i_ap, i_porb, i_tasc, i_f1, i_f0), self.dims)


@dataclass
class Workload:
    name: str
    config_id: int
    P: np.ndarray            # [n_sft][n_bins] fp32
    t_mid: np.ndarray        # [n_sft] fp64 seconds
    vel: np.ndarray          # [n_sft][3] fp64 m/s
    w: np.ndarray            # [n_sft] or [n_sft][n_bins] fp32
    f_min: float
    df: float
    grid: Grid
    stat: str                # "power" | "hough" | "both"
    rho_th: float
    band_width: float
    k: int
    T_sft: float
    planned_injections: list = field(default_factory=list)  # [(template idx tuple, amplitude)]

    @property
    def n_sft(self):
        return self.P.shape[0]

    @property
    def n_bins(self):
        return self.P.shape[1]

    @property
    def per_bin_weights(self) -> bool:
        return self.w.ndim == 2

    @property
    def n_evals(self) -> int:
        return self.grid.n_templates * self.n_sft


# arm-bisector orientation gamma (deg, counter-clockwise from East) of the two LIGO sites, as tabulated with
# the antenna-pattern formulas of the paper's ref. [20]
DETECTOR_GAMMA = {"H1": 171.8, "L1": 243.0, "cfg1": 171.8}


def antenna_geometry(wl: "Workload"):
    """Per-SFT detector geometry for sky-dependent weights (Eq. 4): latitude, arm orientation gamma
    and local sidereal angle at the SFT mid-time (the same rotation phase as earth_velocity), radians.  Rows are
    detector-major (first half H1, second half L1) for the two-detector configs, config 1 is one detector.
    Inputs only: no antenna function is evaluated here."""
    n = wl.n_sft
    names = ["cfg1"] * n if wl.config_id == 1 else ["H1"] * (n - n // 2) + ["L1"] * (n // 2)
    lat = np.array([math.radians(DETECTORS[d][0]) for d in names])
    gam = np.array([math.radians(DETECTOR_GAMMA[d]) for d in names])
    lon = np.array([math.radians(DETECTORS[d][1]) for d in names])
    lst = np.mod(2.0 * math.pi * np.asarray(wl.t_mid, dtype=np.float64) / 86164.0905 + lon, 2.0 * math.pi)
    return lat, gam, lst


def inject(P: np.ndarray, bins: np.ndarray, amplitude: float) -> None:
    """Add `amplitude` at P[alpha][bins[alpha]] for every row (in place).  The bins come from
    the caller (tests: the oracle's track); nothing of the track is computed here."""
    rows = np.arange(P.shape[0])
    P[rows, np.asarray(bins, dtype=np.int64)] += np.float32(amplitude)


def _padding(f_hi, T_sft, max_ap_omega, f1_abs_max, T_span):
    dopp = math.ceil(f_hi * T_sft * (1.0068e-4 + max_ap_omega))
    spin = math.ceil(f1_abs_max * T_span * T_sft) if f1_abs_max > 0 else 0
    return dopp + spin + 2, dopp + 2


def _round4(n):
    return (n + 3) // 4 * 4


def _two_detector_times(config_id, n_sft, T_sft, days, duty=0.7):
    n_slots = int(days * 86400.0 / T_sft)
    rm, rs = _rng(config_id, _S_DUTY), _rng(config_id, _S_SUB)
    per = [n_sft - n_sft // 2, n_sft // 2]
    t, v = [], []
    for det, n_keep in zip(("H1", "L1"), per):
        slots = duty_cycle_slots(rm, rs, n_slots, n_keep, duty)
        tm = (slots.astype(np.float64) + 0.5) * T_sft
        t.append(tm)
        v.append(earth_velocity(tm, *DETECTORS[det]))
    return np.concatenate(t), np.concatenate(v, axis=0)  # detector-major, time-ascending


def config1(n_sky: int = 10) -> Workload:
    """BASELINE.json configs[0]: tiny isolated search, both statistics."""
    cid, T_sft, n_sft = 1, 1800.0, 100
    df = 1.0 / T_sft
    pad, n_band = 60, 180
    n_bins = n_band + 2 * pad
    f_min = 100.0 - pad * df
    t_mid = (np.arange(n_sft, dtype=np.float64) + 0.5) * T_sft
    vel = earth_velocity(t_mid, *DETECTORS["cfg1"])
    P = exponential_spectrogram(_rng(cid, _S_P), n_sft, n_bins)
    w = np.full(n_sft, 1.0 / n_sft, dtype=np.float32)
    grid = Grid(f0_start=100.0, df0=df, n_f0=n_band, sky=fibonacci_sphere(n_sky))
    inj = [((min(3, n_sky - 1), 0, 0, 0, 0, 90), 2.0)]
    return Workload("cfg1-tiny-isolated", cid, P, t_mid, vel, w, f_min, df, grid, "both", 1.6,
                    0.01, 5, T_sft, inj)


def config2(n_sft: int = 4000, n_sky: int = 20000, band_hz: float = 1.0, f_lo: float = 200.0,
            n_f1: int = 5, days: float = 330.0, config_id: int = 2,
            band_width: float = 0.05, k: int = 10) -> Workload:
    """BASELINE.json configs[1] (and the configs[4] sweep through its arguments): isolated
    all-sky, per-SFT noise-floor weights, weighted normalized power."""
    T_sft = 1800.0
    df = 1.0 / T_sft
    n_band = int(round(band_hz * T_sft))
    f1_lo = -1e-9
    t_mid, vel = _two_detector_times(config_id, n_sft, T_sft, days)
    pad_lo, pad_hi = _padding(f_lo + band_hz, T_sft, 0.0, abs(f1_lo), days * 86400.0)
    n_bins = _round4(pad_lo + n_band + pad_hi)
    f_min = f_lo - pad_lo * df
    P = exponential_spectrogram(_rng(config_id, _S_P), n_sft, n_bins)
    r = _rng(config_id, _S_PSD)
    u1, u2 = _uniform_open(r, n_sft), _uniform_open(r, n_sft)
    S = np.exp(0.3 * np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2))  # LogNormal(0,0.3)
    w64 = (1.0 / S) / np.sum(1.0 / S)
    df1 = (0.0 - f1_lo) / (n_f1 - 1) if n_f1 > 1 else 0.0
    grid = Grid(f0_start=f_lo, df0=df, n_f0=n_band, f1_start=f1_lo if n_f1 > 1 else 0.0,
                df1=df1, n_f1=n_f1, sky=fibonacci_sphere(n_sky))
    return Workload(f"cfg{config_id}-allsky-isolated", config_id, P, t_mid, vel,
                    w64.astype(np.float32), f_min, df, grid, "power", 1.6, band_width, k, T_sft)


def config3(n_sft: int = 8000, n_ap: int = 64, n_porb: int = 64, n_tasc: int = 32,
            n_inj: int = 20) -> Workload:
    """BASELINE.json configs[2]: circular-binary search at a fixed sky point, both statistics."""
    cid, T_sft, days = 3, 900.0, 180.0
    df = 1.0 / T_sft
    f_lo, band_hz = 150.0, 0.5
    n_band = int(round(band_hz * T_sft))
    t_mid, vel = _two_detector_times(cid, n_sft, T_sft, days)
    a_p = np.linspace(1.0, 10.0, n_ap)
    P_orb = np.linspace(10.0, 60.0, n_porb) * 86400.0
    tasc = np.arange(n_tasc, dtype=np.float64) / n_tasc
    max_ap_omega = float(a_p.max() * 2.0 * math.pi / P_orb.min())
    pad_lo, pad_hi = _padding(f_lo + band_hz, T_sft, max_ap_omega, 0.0, days * 86400.0)
    n_bins = _round4(pad_lo + n_band + pad_hi)
    f_min = f_lo - pad_lo * df
    P = exponential_spectrogram(_rng(cid, _S_P), n_sft, n_bins)
    w = np.full(n_sft, 1.0 / n_sft, dtype=np.float32)
    ra, dec = 1.0, 0.5
    sky = np.array([[math.cos(dec) * math.cos(ra), math.cos(dec) * math.sin(ra), math.sin(dec)]])
    grid = Grid(f0_start=f_lo, df0=df, n_f0=n_band, sky=sky, a_p=a_p, P_orb=P_orb, tasc_frac=tasc)
    r = _rng(cid, _S_INJ)
    inj = []
    for j in range(n_inj):
        idx = (0, int(r.integers(n_ap)), int(r.integers(n_porb)), int(r.integers(n_tasc)), 0,
               int(r.integers(n_band)))
        inj.append((idx, 0.5 + 2.5 * j / max(1, n_inj - 1)))
    return Workload("cfg3-binary-fixed-sky", cid, P, t_mid, vel, w, f_min, df, grid, "both", 1.6,
                    0.01, 10, T_sft, inj)


def config4(n_sft: int = 6000, n_sky: int = 5000, band_hz: float = 2.0, n_lines: int = 30) -> Workload:
    """BASELINE.json configs[3]: non-stationary lines, per-bin weights w[alpha][k] = 1/S_{alpha,k}
    normalised per bin (reading R18: each line bin is loud in one contiguous epoch
    covering half the SFTs, PSD multiplier 20)."""
    cid, T_sft, days = 4, 1800.0, 330.0
    df = 1.0 / T_sft
    f_lo = 50.0
    n_band = int(round(band_hz * T_sft))
    f1_lo, n_f1 = -1e-9, 3
    t_mid, vel = _two_detector_times(cid, n_sft, T_sft, days)
    pad_lo, pad_hi = _padding(f_lo + band_hz, T_sft, 0.0, abs(f1_lo), days * 86400.0)
    n_bins = _round4(pad_lo + n_band + pad_hi)
    f_min = f_lo - pad_lo * df
    P = exponential_spectrogram(_rng(cid, _S_P), n_sft, n_bins)
    r = _rng(cid, _S_PSD)
    u1, u2 = _uniform_open(r, n_sft), _uniform_open(r, n_sft)
    S_alpha = np.exp(0.3 * np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2))
    mult = np.ones((n_sft, n_bins), dtype=np.float64)
    rl = _rng(cid, _S_LINES)
    line_bins = rl.permutation(n_bins)[:n_lines]
    half = n_sft // 2
    for kb in line_bins:
        start = int(rl.integers(0, n_sft - half + 1))
        mult[start:start + half, kb] = 20.0
    P *= mult.astype(np.float32)
    inv_S = 1.0 / (S_alpha[:, None] * mult)
    w = (inv_S / inv_S.sum(axis=0, keepdims=True)).astype(np.float32)
    grid = Grid(f0_start=f_lo, df0=df, n_f0=n_band, f1_start=f1_lo, df1=-f1_lo / (n_f1 - 1),
                n_f1=n_f1, sky=fibonacci_sphere(n_sky))
    return Workload("cfg4-lines-per-bin-weights", cid, P, t_mid, vel, w, f_min, df, grid, "power",
                    1.6, 0.1, 20, T_sft)


# BASELINE.json configs[4]: the sweeps.  (n_sft, band Hz, n_sky)
SWEEP_A = [(500, 0.1, 1112), (2000, 0.5, 2223), (8000, 1.0, 11112), (8000, 2.0, 55556),
           (16000, 4.0, 277778)]
SWEEP_B = [(n, 1.0, 11112) for n in (500, 2000, 8000, 16000)]


def config5(n_sft: int, band_hz: float, n_sky: int) -> Workload:
    return config2(n_sft=n_sft, n_sky=n_sky, band_hz=band_hz, config_id=5)


def by_id(config_id: int, **kw) -> Workload:
    return {1: config1, 2: config2, 3: config3, 4: config4}[config_id](**kw)


TEMPLATE_DTYPE = np.dtype([("f0", "<f8"), ("f1", "<f8"), ("nx", "<f8"), ("ny", "<f8"), ("nz", "<f8"),
                           ("a_p", "<f8"), ("P_orb", "<f8"), ("t_asc", "<f8")])


def random_bank(wl: Workload, n: int, seed: int = 0) -> np.ndarray:
    """Unstructured template bank (PAPER.md:312-316 draws banks at random over the parameter space;
    here uniformly over the physical box the workload's grid spans, a stand-in for the paper's
    uniform draw in the xi coordinates of Eq. A11): n records (f0, f1, n, a_p, P_orb, t_asc).
    f0 uniform over the grid's band, f1 over its spindown range, sky isotropic when the grid is
    all-sky (else the grid's point), orbit uniform over the grid's a_p / P_orb ranges, t_asc over
    one orbit after t_ref.  Parameters only: no track, no statistic."""
    g = wl.grid
    rng = np.random.Generator(np.random.PCG64((BASE_SEED + wl.config_id) * 16 + 8 + 16 * seed))
    tl = np.zeros(n, dtype=TEMPLATE_DTYPE)
    tl["f0"] = g.f0_start + rng.random(n) * (g.n_f0 - 1) * g.df0
    f1_hi = g.f1_start + (g.n_f1 - 1) * g.df1
    tl["f1"] = g.f1_start + rng.random(n) * (f1_hi - g.f1_start)
    if len(g.sky) > 1:
        z = 2.0 * rng.random(n) - 1.0
        phi = 2.0 * math.pi * rng.random(n)
        r = np.sqrt(1.0 - z * z)
        tl["nx"], tl["ny"], tl["nz"] = r * np.cos(phi), r * np.sin(phi), z
    else:
        tl["nx"], tl["ny"], tl["nz"] = g.sky[0]
    a_lo, a_hi = float(np.min(g.a_p)), float(np.max(g.a_p))
    p_lo, p_hi = float(np.min(g.P_orb)), float(np.max(g.P_orb))
    tl["a_p"] = a_lo + rng.random(n) * (a_hi - a_lo)
    tl["P_orb"] = p_lo + rng.random(n) * (p_hi - p_lo)
    tl["t_asc"] = g.t_ref + rng.random(n) * tl["P_orb"]
    return tl
