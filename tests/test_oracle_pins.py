"""Pins of the CPU oracle (oracle/ft_oracle.c) against what the paper and the mathematics fix.

The paper prints no worked numeric example (PAPER.md has no input/output pair for Eq. 3), so every
pin is a closed form, an invariant, a special case that reduces to a library routine, an exact /
50-digit evaluation, or brute force on tiny inputs.  Each test says which mistake it would catch.
"""
import math
from fractions import Fraction

import mpmath
import numpy as np
import pytest

from oracle import ft_oracle as fo
from paper_2411_18370_b200 import workloads as W


def _simple_workload(n_sft=64, n_bins=256, df=1.0 / 1800.0, f_lo=100.0, pad=40, n_f0=None, seed=7,
                     vel=None, grid_kw=None, w=None, P=None, t_mid=None):
    rng = np.random.Generator(np.random.PCG64(seed))
    T = 1.0 / df
    t_mid = (np.arange(n_sft) + 0.5) * T if t_mid is None else t_mid
    vel = W.earth_velocity(t_mid, 46.45, 0.0) if vel is None else vel
    P = (-np.log(1.0 - rng.random((n_sft, n_bins)))).astype(np.float32) if P is None else P
    w = np.full(n_sft, 1.0 / n_sft, np.float32) if w is None else w
    n_f0 = n_bins - 2 * pad if n_f0 is None else n_f0
    g = dict(f0_start=f_lo, df0=df, n_f0=n_f0)
    g.update(grid_kw or {})
    return W.Workload("t", 99, P, t_mid, vel, w, f_lo - pad * df, df, W.Grid(**g), "both", 1.6,
                      0.01, 5, T)


# ---------------------------------------------------------------- T1: Eq. (13)-(14) noise moments
def test_noise_mean_and_variance_eq13_eq14(golden):
    """Catches: a dropped weight, wrong normalisation, gathering the same pixel twice."""
    wl = W.config2(n_sft=400, n_sky=3)
    o = fo.Oracle(wl)
    n_f0 = wl.grid.n_f0
    power = o.eval_range(0, n_f0)[0]          # one sky point, one f1: disjoint columns -> independent
    w = wl.w.astype(np.float64)
    mean_th = golden["noise_mean_per_sum_w_exp1"] * w.sum()
    var_th = golden["noise_var_per_sum_w2_exp1"] * (w ** 2).sum()
    se = math.sqrt(var_th / n_f0)
    assert abs(power.mean() - mean_th) < 4 * se
    assert abs(power.var() / var_th - 1.0) < 4 * math.sqrt(2.0 / n_f0) + 0.05
    # chi^2_2 scale of the paper: multiply pixels by 2 -> mu_G = 2 sum w (Eq. 13)
    wl2 = W.config2(n_sft=400, n_sky=3)
    wl2.P *= np.float32(2.0)
    p2 = fo.Oracle(wl2).eval_range(0, n_f0)[0]
    assert abs(p2.mean() - golden["noise_mean_per_sum_w_chi2"] * w.sum()) < 8 * se


# ---------------------------------------------------------------- T2: Eq. (7), (11) binomial count
def test_hough_count_is_binomial(golden):
    """Catches: >= instead of >, threshold on the wrong scale, count not integer/in range."""
    wl = W.config2(n_sft=400, n_sky=3)
    o = fo.Oracle(wl, rho_th=golden["hough_threshold_exp1"])
    n_f0, n = wl.grid.n_f0, wl.n_sft
    _, cnt, wcnt, _ = o.eval_range(0, n_f0)
    p = golden["hough_p"]
    assert p == pytest.approx(math.exp(-golden["hough_threshold_chi2"] / 2.0), rel=1e-15)
    assert cnt.min() >= 0 and cnt.max() <= n
    assert abs(cnt.mean() - n * p) < 4 * math.sqrt(n * p * (1 - p) / n_f0)
    assert abs(cnt.var() / (n * p * (1 - p)) - 1.0) < 4 * math.sqrt(2.0 / n_f0) + 0.05
    # weighted count: mean = p * sum w (Eq. 3 applied to Eq. 7)
    w = wl.w.astype(np.float64)
    assert abs(wcnt.mean() - p * w.sum()) < 4 * math.sqrt(p * (1 - p) * (w ** 2).sum() / n_f0)
    # non-increasing in rho_th; strict '>' : threshold equal to a pixel value excludes it
    c_lo = fo.Oracle(wl, rho_th=1.0).eval_range(0, n_f0)[1]
    c_hi = fo.Oracle(wl, rho_th=2.5).eval_range(0, n_f0)[1]
    assert np.all(c_lo >= cnt) and np.all(cnt >= c_hi)


def test_hough_strict_greater_than():
    P = np.full((8, 64), 1.6, np.float32)   # (float)1.6 == pixel -> not counted (strict >)
    wl = _simple_workload(n_sft=8, n_bins=64, pad=20, P=P)
    assert np.all(fo.Oracle(wl, rho_th=1.6).eval_range()[1] == 0)
    assert np.all(fo.Oracle(wl, rho_th=np.nextafter(np.float32(1.6), np.float32(0))).eval_range()[1] == 8)


# ---------------------------------------------------------------- T3: a_p = 0 is the isolated track
def test_ap_zero_reduces_to_isolated():
    """PAPER.md:56 'For a_p = 0 the source effectively behaves like an isolated one'."""
    base = _simple_workload(grid_kw=dict(sky=W.fibonacci_sphere(4)))
    iso = fo.Oracle(base).eval_range()
    binw = _simple_workload(grid_kw=dict(sky=W.fibonacci_sphere(4), a_p=np.array([0.0, 3.0]),
                                         P_orb=np.array([5.0, 9.0]) * 86400.0,
                                         tasc_frac=np.array([0.0, 0.37])))
    ob = fo.Oracle(binw)
    full = ob.eval_range()
    dims = ob.dims
    pw = full[0].reshape(dims)
    ct = full[1].reshape(dims)
    iso_pw = iso[0].reshape(4, 1, 1, 1, 1, -1)
    for ip in range(2):
        for it in range(2):
            assert np.array_equal(pw[:, 0, ip, it], iso_pw[:, 0, 0, 0])
            assert np.array_equal(ct[:, 0, ip, it], iso[1].reshape(4, 1, 1, 1, 1, -1)[:, 0, 0, 0])
    assert not np.array_equal(pw[:, 1, 0, 0], iso_pw[:, 0, 0, 0])  # a_p = 3 does move the track


# ---------------------------------------------------------------- T4: straight line = column sum
def test_zero_velocity_is_weighted_column_sum():
    """v = 0, a_p = 0, f1 = 0: s(f0_i) = sum_alpha w_alpha P[alpha][pad + i] — a GEMV (w^T P).
    Catches: transposed spectrogram, off-by-one in the bin origin, weight index mix-up."""
    n_sft, n_bins, pad = 50, 200, 30
    rng = np.random.Generator(np.random.PCG64(3))
    w = rng.random(n_sft).astype(np.float32)
    wl = _simple_workload(n_sft=n_sft, n_bins=n_bins, pad=pad, vel=np.zeros((n_sft, 3)), w=w)
    pw, ct, wc, _ = fo.Oracle(wl).eval_range()
    ref = w.astype(np.float64) @ wl.P.astype(np.float64)
    assert np.allclose(pw, ref[pad:n_bins - pad], rtol=1e-13, atol=0)
    assert np.array_equal(ct, (wl.P > np.float32(1.6)).sum(0)[pad:n_bins - pad])
    refc = w.astype(np.float64) @ (wl.P > np.float32(1.6)).astype(np.float64)
    assert np.allclose(wc, refc[pad:n_bins - pad], rtol=1e-13)
    # per-bin weights: same reduction with w[alpha][k]
    w2 = rng.random((n_sft, n_bins)).astype(np.float32)
    wl2 = _simple_workload(n_sft=n_sft, n_bins=n_bins, pad=pad, vel=np.zeros((n_sft, 3)), w=w2)
    pw2 = fo.Oracle(wl2).eval_range()[0]
    ref2 = (w2.astype(np.float64) * wl2.P.astype(np.float64)).sum(0)
    assert np.allclose(pw2, ref2[pad:n_bins - pad], rtol=1e-13)


# ---------------------------------------------------------------- T5: injected track
def test_injected_track_recovers_exact_sum():
    """Eq. (3) on a noiseless spectrogram with amplitude A along lambda*: s = A sum w, count = n_sft,
    mismatch m(lambda*; lambda*) = 0 (Eq. 24); every other template scores <= that."""
    n_sft = 80
    g = dict(sky=W.fibonacci_sphere(5), a_p=np.array([0.0, 2.0, 4.0]),
             P_orb=np.array([3.0, 4.5]) * 86400.0, tasc_frac=np.array([0.1, 0.6]))
    rng = np.random.Generator(np.random.PCG64(11))
    w = (rng.random(n_sft) + 0.5).astype(np.float32)
    wl = _simple_workload(n_sft=n_sft, n_bins=256, pad=40, grid_kw=g, w=w,
                          P=np.zeros((n_sft, 256), np.float32))
    o = fo.Oracle(wl)
    star = int(wl.grid.ravel(3, 2, 1, 1, 0, 77))
    k, _, rc = o.track(star)
    assert rc == 0
    A = 2.0
    W.inject(wl.P, k, A)
    o = fo.Oracle(wl)
    pw, ct, _, _ = o.eval_range()
    assert pw[star] == pytest.approx(A * w.astype(np.float64).sum(), rel=1e-14)
    assert ct[star] == n_sft
    assert np.all(pw <= pw[star]) and np.all(ct <= n_sft)
    mu_g = 0.0  # noiseless
    assert (pw[star] - pw[star]) / (pw[star] - mu_g) == 0.0   # Eq. (24) at the true template


# ---------------------------------------------------------------- T6: one-bin resolution, Eq. (27)
def test_resolution_property_eq27_eqA1_eq28():
    """delta f0 = 1/T_SFT (Eq. A1) moves every bin by 1 (0 or 2 only across a rounding boundary);
    delta a_p = 1/(T_SFT f0 Omega) and delta phi_b = 1/(T_SFT f0 a_p Omega) (Eq. 28) move the
    track by about one bin at most.  Catches: wrong units of a_p/Omega, missing factor f0."""
    T, f0 = 900.0, 150.0
    n_sft = 960
    t_mid = (np.arange(n_sft) + 0.5) * T
    P_orb, a_p = 10.0 * T * 96, 8.0         # 10 days in units of T_SFT
    Om = 2 * math.pi / P_orb
    d_ap = 1.0 / (T * f0 * Om)
    d_phi = 1.0 / (T * f0 * a_p * Om)       # radians; as a t_asc fraction: d_phi / (2 pi)
    g = dict(f0_start=f0, df0=1.0 / T, n_f0=3, a_p=np.array([a_p, a_p + d_ap]),
             P_orb=np.array([P_orb]), tasc_frac=np.array([0.25, 0.25 + d_phi / (2 * math.pi)]))
    wl = _simple_workload(n_sft=n_sft, n_bins=400, df=1.0 / T, f_lo=f0, pad=150, t_mid=t_mid,
                          grid_kw=g)
    o = fo.Oracle(wl)
    k000 = o.track(int(wl.grid.ravel(0, 0, 0, 0, 0, 0)))[0]
    k_f0 = o.track(int(wl.grid.ravel(0, 0, 0, 0, 0, 1)))[0]
    k_ap = o.track(int(wl.grid.ravel(0, 1, 0, 0, 0, 0)))[0]
    k_ph = o.track(int(wl.grid.ravel(0, 0, 0, 1, 0, 0)))[0]
    d = k_f0 - k000
    assert set(np.unique(d)) <= {0, 1, 2} and (d == 1).mean() > 0.99
    for kk in (k_ap, k_ph):
        assert 1 <= np.abs(kk - k000).max() <= 2
    # a 10x finer step than the resolution leaves most of the track unchanged
    g2 = dict(g, a_p=np.array([a_p, a_p + 0.1 * d_ap]))
    wl2 = _simple_workload(n_sft=n_sft, n_bins=400, df=1.0 / T, f_lo=f0, pad=150, t_mid=t_mid,
                           grid_kw=g2)
    o2 = fo.Oracle(wl2)
    same = o2.track(int(wl2.grid.ravel(0, 1, 0, 0, 0, 0)))[0] == o2.track(0)[0]
    assert same.mean() > 0.85


# ---------------------------------------------------------------- closed-form binary extremes
def test_binary_track_extremes_and_period():
    """At v = 0 the track is f0 [1 - a_p Omega cos(Omega (t - t_asc))] (Eq. 2): its extreme bins are
    rint((f0 (1 -+ a_p Omega) - f_min)/df) and the bin sequence has period P_orb on a gap-free grid.
    Catches: sin for cos, wrong sign of the binary term, Omega = P/2pi, t_asc not t_ref + u P."""
    T = 900.0
    per = 64                                   # P_orb = 64 T_SFT
    n_sft = 4 * per
    t_mid = (np.arange(n_sft) + 0.5) * T
    P_orb, a_p, f0, u = per * T, 40.0, 150.0, 0.5 / per  # t_asc = t_mid[0]
    g = dict(f0_start=f0, df0=1.0 / T, n_f0=2, a_p=np.array([a_p]), P_orb=np.array([P_orb]),
             tasc_frac=np.array([u]))
    wl = _simple_workload(n_sft=n_sft, n_bins=1200, df=1.0 / T, f_lo=f0, pad=590, t_mid=t_mid,
                          vel=np.zeros((n_sft, 3)), grid_kw=g)
    k, x, rc = fo.Oracle(wl).track(0)
    assert rc == 0
    Om = 2 * math.pi / P_orb
    lo = round((f0 * (1 - a_p * Om) - wl.f_min) * T)
    hi = round((f0 * (1 + a_p * Om) - wl.f_min) * T)
    assert k[0] == lo == k.min()               # cos(0) = 1 at t = t_asc: minimum frequency
    assert k[per // 2] == hi == k.max()        # half an orbit later: maximum
    assert hi - lo > 300                       # the modulation is resolved (not a trivial pass)
    assert np.array_equal(k[:-per], k[per:])   # period P_orb
    assert not np.array_equal(k[:-per // 2], k[per // 2:])


# ---------------------------------------------------------------- exact-rational track (isolated)
def _half_even(fr: Fraction) -> int:
    fl = math.floor(fr)
    r = fr - fl
    if r > Fraction(1, 2) or (r == Fraction(1, 2) and fl % 2 == 1):
        return fl + 1
    return fl


def test_isolated_track_against_exact_rational_arithmetic():
    """Evaluate Eq. (2) (with f1) in exact rational arithmetic from the same double inputs; the
    fp64 oracle must give the same bin except within 1e-9 of a tie, and x within 1e-9.
    Catches: any dropped term, sign, operand or index error in the track."""
    wl = W.config2(n_sft=120, n_sky=7)
    o = fo.Oracle(wl)
    g = wl.grid
    rng = np.random.Generator(np.random.PCG64(5))
    c = Fraction(299792458)
    for idx in rng.integers(0, g.n_templates, 12):
        i_sky, _, _, _, i_f1, i_f0 = (int(v) for v in g.unravel(idx))
        k, x, rc = o.track(int(idx))
        assert rc == 0
        f0 = Fraction(g.f0_start) + i_f0 * Fraction(g.df0)
        f1 = Fraction(g.f1_start) + i_f1 * Fraction(g.df1)
        n = [Fraction(float(v)) for v in g.sky[i_sky]]
        for a in range(0, wl.n_sft, 7):
            t = Fraction(float(wl.t_mid[a]))
            V = sum(Fraction(float(wl.vel[a, j])) * n[j] for j in range(3)) / c
            xe = ((f0 + f1 * (t - Fraction(g.t_ref))) * (1 + V) - Fraction(wl.f_min)) / Fraction(wl.df)
            assert abs(float(xe) - x[a]) < 1e-9
            if abs((xe - math.floor(xe)) - Fraction(1, 2)) > Fraction(1, 10 ** 8):
                assert _half_even(xe) == k[a]


def test_binary_track_against_50_digit_evaluation():
    """Same as above with the binary term, in 50-digit mpmath (true pi, true cos)."""
    mpmath.mp.dps = 50
    wl = W.config3(n_sft=200, n_ap=5, n_porb=4, n_tasc=3, n_inj=0)
    o = fo.Oracle(wl)
    g = wl.grid
    rng = np.random.Generator(np.random.PCG64(6))
    mpf = mpmath.mpf
    for idx in rng.integers(0, g.n_templates, 10):
        i_sky, i_ap, i_po, i_ta, _, i_f0 = (int(v) for v in g.unravel(idx))
        k, x, rc = o.track(int(idx))
        assert rc == 0
        f0 = mpf(g.f0_start) + i_f0 * mpf(g.df0)
        Om = 2 * mpmath.pi / mpf(float(g.P_orb[i_po]))
        t_asc = mpf(g.t_ref) + mpf(float(g.tasc_frac[i_ta])) * mpf(float(g.P_orb[i_po]))
        n = [mpf(float(v)) for v in g.sky[i_sky]]
        for a in range(0, wl.n_sft, 5):
            t = mpf(float(wl.t_mid[a]))
            V = sum(mpf(float(wl.vel[a, j])) * n[j] for j in range(3)) / mpf(299792458)
            B = mpf(float(g.a_p[i_ap])) * Om * mpmath.cos(Om * (t - t_asc))
            xe = (f0 * (1 + V - B) - mpf(wl.f_min)) / mpf(wl.df)
            assert abs(xe - mpf(float(x[a]))) < mpf(10) ** -9
            if abs((xe - mpmath.floor(xe)) - mpf(1) / 2) > mpf(10) ** -8:
                assert int(mpmath.nint(xe)) == k[a]


# ---------------------------------------------------------------- rounding mode (reading R5)
def test_round_half_to_even_and_near_tie_flag():
    n_sft, n_bins = 4, 16
    P = np.arange(n_sft * n_bins, dtype=np.float32).reshape(n_sft, n_bins)
    t_mid = np.arange(n_sft) + 0.5
    for f0, k_expect in ((2.5, 2), (3.5, 4), (4.5, 4), (2.25, 2), (2.75, 3)):
        wl = W.Workload("r", 99, P, t_mid, np.zeros((n_sft, 3)), np.ones(n_sft, np.float32), 0.0, 1.0,
                        W.Grid(f0_start=f0, df0=1.0, n_f0=1), "both", 1.6, 1.0, 1, 1.0)
        o = fo.Oracle(wl)
        k, x, _ = o.track(0)
        assert np.all(k == k_expect) and np.all(x == f0)
        tie = o.eval_range()[3][0]
        assert tie == (1 if f0 % 1 == 0.5 else 0)
        assert o.eval_range()[0][0] == P[:, k_expect].astype(np.float64).sum()


def test_track_out_of_range_is_an_error():
    wl = _simple_workload(n_sft=8, n_bins=64, pad=0)    # no Doppler padding: tracks leave the band
    o = fo.Oracle(wl)
    with pytest.raises(ValueError):
        o.eval_range()


# ---------------------------------------------------------------- T7: metamorphic
def test_linearity_and_permutation_invariance():
    wl = W.config2(n_sft=160, n_sky=4)
    o = fo.Oracle(wl)
    pw, ct, wc, _ = o.eval_range(0, 3000)
    wl2 = W.config2(n_sft=160, n_sky=4)
    wl2.P *= np.float32(2.0)                       # exact scaling
    pw2 = fo.Oracle(wl2).eval_range(0, 3000)[0]
    assert np.array_equal(pw2, 2.0 * pw)
    perm = np.random.Generator(np.random.PCG64(1)).permutation(wl.n_sft)
    wl3 = W.config2(n_sft=160, n_sky=4)
    wl3.P, wl3.t_mid, wl3.vel, wl3.w = wl3.P[perm], wl3.t_mid[perm], wl3.vel[perm], wl3.w[perm]
    pw3, ct3, wc3, _ = fo.Oracle(wl3).eval_range(0, 3000)
    assert np.array_equal(ct3, ct)                 # integer counts: exact under SFT reordering
    assert np.allclose(pw3, pw, rtol=1e-13) and np.allclose(wc3, wc, rtol=1e-13)


# ---------------------------------------------------------------- T8: brute force on tiny inputs
def test_brute_force_python_on_tiny_grid():
    """Independent nested-loop Python evaluation (index order by explicit loops, Python floats,
    round() = half-even).  Catches: canonical index order / unravel mistakes, list vs range API."""
    n_sft = 11
    g = dict(n_f0=7, f1_start=-2e-9, df1=1e-9, n_f1=2, sky=W.fibonacci_sphere(3),
             a_p=np.array([0.0, 1.5]), P_orb=np.array([1.0, 2.5]) * 86400.0,
             tasc_frac=np.array([0.0, 0.4]))
    wl = _simple_workload(n_sft=n_sft, n_bins=96, pad=40, grid_kw=g, n_f0=7)
    wl.grid.f0_start, wl.grid.df0 = 100.0, wl.df
    o = fo.Oracle(wl)
    pw, ct, wc, _ = o.eval_range()
    idx = 0
    for sky in wl.grid.sky:
        for ap in wl.grid.a_p:
            for Po in wl.grid.P_orb:
                for u in wl.grid.tasc_frac:
                    for j in range(2):
                        for i in range(7):
                            f0 = 100.0 + i * wl.df
                            f1 = -2e-9 + j * 1e-9
                            Om = 6.283185307179586 / Po
                            tasc = 0.0 + u * Po
                            s, c = 0.0, 0
                            for a in range(n_sft):
                                t = float(wl.t_mid[a])
                                V = ((wl.vel[a, 0] * sky[0] + wl.vel[a, 1] * sky[1]) + wl.vel[a, 2] * sky[2]) / 299792458.0
                                B = (ap * Om) * math.cos(Om * (t - tasc)) if ap != 0.0 else 0.0
                                x = (((f0 + f1 * (t - 0.0)) * ((1.0 + V) - B)) - wl.f_min) * (1.0 / wl.df)
                                k = round(x)
                                p = wl.P[a, k]
                                s += float(wl.w[a]) * float(p)
                                c += int(p > np.float32(1.6))
                            assert pw[idx] == s and ct[idx] == c, idx
                            idx += 1
    assert idx == o.n_templates
    sub = np.array([5, 0, 111, 77, o.n_templates - 1], dtype=np.uint64)
    lp, lc, lw, _ = o.eval_list(sub)
    assert np.array_equal(lp, pw[sub.astype(np.int64)]) and np.array_equal(lc, ct[sub.astype(np.int64)])
    rp = o.eval_range(70, 90)[0]
    assert np.array_equal(rp, pw[70:90])


def test_topk_per_band_is_exhaustive_sort():
    """Brute force with Python's sorted() on config 1 (T8): (value desc, index asc), k per band."""
    wl = W.config1()
    o = fo.Oracle(wl)
    pw, ct, _, _ = o.eval_range()
    n_f0, bpb, k = wl.grid.n_f0, 18, 5
    for vals in (pw, ct):
        got = fo.topk_per_band(vals, n_f0, bpb, k)
        assert len(got) == 10
        for b, (gi, gv) in enumerate(got):
            members = [(-float(vals[j]), j) for j in range(vals.size) if (j % n_f0) // bpb == b]
            ref = sorted(members)[:k]
            assert [j for _, j in ref] == [int(v) for v in gi]
            assert [-v for v, _ in ref] == [float(v) for v in gv]


def test_config1_injection_is_loudest_in_its_band():
    wl = W.config1()
    (tidx, amp), = wl.planned_injections
    star = int(wl.grid.ravel(*tidx))
    k, _, _ = fo.Oracle(wl).track(star)
    before = fo.Oracle(wl).eval_range()[0]
    W.inject(wl.P, k, amp)
    after = fo.Oracle(wl).eval_range()[0]
    assert after[star] == pytest.approx(before[star] + amp * float(wl.w.astype(np.float64).sum()), rel=1e-6)  # fp32 pixels
    top = fo.topk_per_band(after, wl.grid.n_f0, 18, 5)
    assert int(top[90 // 18][0][0]) == star


# ------------------------------------------------- unstructured banks (explicit template lists)
def _explicit_from_grid(wl):
    """Every grid template written out as an explicit (f0, f1, n, a_p, P_orb, t_asc) record, in
    canonical order, by plain loops (no oracle code)."""
    g = wl.grid
    recs = []
    for sky in g.sky:
        for ap in g.a_p:
            for Po in g.P_orb:
                for u in g.tasc_frac:
                    for j in range(g.n_f1):
                        for i in range(g.n_f0):
                            recs.append((g.f0_start + i * g.df0, g.f1_start + j * g.df1, sky[0], sky[1], sky[2],
                                         ap, Po, g.t_ref + u * Po))
    return np.array(recs, dtype=fo.TEMPLATE_DTYPE)


def test_template_list_reproduces_the_grid_bit_for_bit():
    """An explicit list that enumerates a product grid gives the grid's statistics exactly
    (parameter mapping, t_asc = t_ref + u P_orb, index order)."""
    g = dict(n_f0=9, f1_start=-1e-9, df1=1e-9, n_f1=2, sky=W.fibonacci_sphere(3),
             a_p=np.array([0.0, 2.0]), P_orb=np.array([1.5]) * 86400.0, tasc_frac=np.array([0.25, 0.5]))
    wl = _simple_workload(n_sft=23, n_bins=96, pad=40, grid_kw=g, n_f0=9)
    wl.grid.f0_start, wl.grid.df0 = 100.0, wl.df
    o = fo.Oracle(wl)
    pw, ct, wc, tie = o.eval_range()
    lp, lc, lw, lt = fo.eval_templates(o, _explicit_from_grid(wl), wl.grid.t_ref)
    assert np.array_equal(lp, pw) and np.array_equal(lc, ct) and np.array_equal(lw, wc) and np.array_equal(lt, tie)


def test_template_list_brute_force_off_grid_with_reference_time():
    """Off-grid templates (random f0 between bins, random sky, binary parameters) and t_ref != 0,
    against an independent Python loop.  Catches: t_ref used in the wrong place, t_asc treated as
    a fraction, a swapped field of the record."""
    wl = _simple_workload(n_sft=17, n_bins=96, pad=40, grid_kw={}, n_f0=4)
    rng = np.random.Generator(np.random.PCG64(77))
    n, t_ref = 40, 3000.0
    tl = np.zeros(n, dtype=fo.TEMPLATE_DTYPE)
    tl["f0"] = 100.0 + rng.random(n) * 10 * wl.df
    tl["f1"] = -2e-9 * rng.random(n)
    v = rng.normal(size=(n, 3)); v /= np.linalg.norm(v, axis=1, keepdims=True)
    tl["nx"], tl["ny"], tl["nz"] = v[:, 0], v[:, 1], v[:, 2]
    tl["a_p"] = np.where(rng.random(n) < 0.3, 0.0, 0.3 * rng.random(n))
    tl["P_orb"] = (0.5 + 2.0 * rng.random(n)) * 86400.0
    tl["t_asc"] = 1e5 * rng.random(n)
    o = fo.Oracle(wl)
    pw, ct, wc, _ = fo.eval_templates(o, tl, t_ref)
    for q in range(n):
        f0, f1, nx, ny, nz, ap, Po, tasc = (float(tl[q][k]) for k in fo.TEMPLATE_DTYPE.names)
        Om = 6.283185307179586 / Po
        s, c, sw = 0.0, 0, 0.0
        for a in range(wl.n_sft):
            t = float(wl.t_mid[a])
            V = ((wl.vel[a, 0] * nx + wl.vel[a, 1] * ny) + wl.vel[a, 2] * nz) / 299792458.0
            B = (ap * Om) * math.cos(Om * (t - tasc)) if ap != 0.0 else 0.0
            x = (((f0 + f1 * (t - t_ref)) * ((1.0 + V) - B)) - wl.f_min) * (1.0 / wl.df)
            k = round(x)
            p = wl.P[a, k]
            s += float(wl.w[a]) * float(p)
            if p > np.float32(1.6):
                c += 1
                sw += float(wl.w[a])
        assert pw[q] == s and ct[q] == c and wc[q] == sw, q


def test_template_list_straight_line_is_a_column_sum():
    """v = 0, a_p = 0, f1 = 0 at an OFF-grid f0: the track is the single column rint((f0 - f_min)/df)
    and the statistic is the weighted sum of that column (a GEMV row)."""
    wl = _simple_workload(n_sft=50, n_bins=64, pad=10, grid_kw={}, n_f0=4)
    wl.vel[:] = 0.0
    o = fo.Oracle(wl)
    tl = np.zeros(3, dtype=fo.TEMPLATE_DTYPE)
    tl["nz"], tl["P_orb"] = 1.0, 86400.0
    tl["f0"] = wl.f_min + np.array([12.3, 12.7, 40.49]) * wl.df
    pw, ct, _, _ = fo.eval_templates(o, tl, 0.0)
    colsum = (wl.w.astype(np.float64)[:, None] * wl.P.astype(np.float64))
    for q, col in enumerate([12, 13, 40]):
        assert abs(pw[q] - colsum[:, col].sum()) <= 1e-12 * pw[q]
        assert ct[q] == int((wl.P[:, col] > np.float32(1.6)).sum())


# ---------------------------------------------------------------- near-tie window WIDTH (north_star: 1e-9 bin)
def test_near_tie_window_width():
    """Catches: a window wider or narrower than 1e-9 bin (a 1e-4 window would silently exempt templates from
    parity).  df = 1, f_min = 0, v = 0: x = f0 exactly, so x = k + 0.5 + delta is built by hand."""
    n_sft, n_bins = 3, 256
    P = np.ones((n_sft, n_bins), np.float32)
    t_mid = np.arange(n_sft) + 0.5
    for k in (2, 100, 201):
        for delta, flagged in ((5e-10, 1), (-5e-10, 1), (9e-10, 1), (-9e-10, 1), (2e-9, 0), (-2e-9, 0),
                               (1.1e-9, 0), (-1.1e-9, 0), (1e-4, 0), (-1e-4, 0), (0.25, 0)):
            f0 = k + 0.5 + delta
            wl = W.Workload("w", 99, P, t_mid, np.zeros((n_sft, 3)), np.ones(n_sft, np.float32), 0.0, 1.0,
                            W.Grid(f0_start=f0, df0=1.0, n_f0=1), "both", 1.6, 1.0, 1, 1.0)
            o = fo.Oracle(wl)
            x = o.track(0)[1]
            assert np.all(x == f0)
            assert o.eval_range()[3][0] == flagged, (k, delta)


# ---------------------------------------------------------------- Eq. (4)-(5): antenna-pattern weights
def _detector_tensor_response(lat, gamma, lst, ra, dec):
    """F+^2 + Fx^2 from the geometry alone: detector tensor d = (n1 n1 - n2 n2)/2 of two perpendicular arms at
    gamma -+ 45 deg counter-clockwise from East at (lat, local sidereal angle lst), contracted with the
    polarisation tensors of a wave from (ra, dec).  No formula shared with the oracle."""
    e_east = np.array([-math.sin(lst), math.cos(lst), 0.0])
    e_north = np.array([-math.sin(lat) * math.cos(lst), -math.sin(lat) * math.sin(lst), math.cos(lat)])
    arms = [math.cos(gamma + s * math.pi / 4) * e_east + math.sin(gamma + s * math.pi / 4) * e_north for s in (-1, 1)]
    d = 0.5 * (np.outer(arms[0], arms[0]) - np.outer(arms[1], arms[1]))
    xi = np.array([math.sin(ra), -math.cos(ra), 0.0])
    eta = np.array([-math.sin(dec) * math.cos(ra), -math.sin(dec) * math.sin(ra), math.cos(dec)])
    fp = np.sum(d * (np.outer(xi, xi) - np.outer(eta, eta)))
    fc = np.sum(d * (np.outer(xi, eta) + np.outer(eta, xi)))
    return fp * fp + fc * fc


def test_antenna_functions_against_detector_tensor_and_sky_average(golden):
    """Catches: a wrong coefficient, sign or angle in a(t), b(t) (ref. [20] Eq. 12-13): a^2 + b^2 must equal
    F+^2 + Fx^2 of the detector tensor for perpendicular arms, for any detector, time and source."""
    rng = np.random.Generator(np.random.PCG64(42))
    for _ in range(300):
        lat, gamma, lst = rng.uniform(-1.5, 1.5), rng.uniform(0, 2 * math.pi), rng.uniform(0, 2 * math.pi)
        ra, dec = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-1, 1))
        a, b = fo.antenna_ab(lat, gamma, lst, ra, dec)
        assert abs((a * a + b * b) - _detector_tensor_response(lat, gamma, lst, ra, dec)) < 1e-12
    # sky average 2/5 (Gauss-Legendre in sin(dec), uniform in ra: exact for the degree-4 polynomial integrand)
    xs, ws = np.polynomial.legendre.leggauss(8)
    ras = (np.arange(16) + 0.5) * 2 * math.pi / 16
    for lat, gamma, lst in ((0.81, 2.99, 0.3), (0.53, 4.24, 5.0), (-0.2, 0.0, 1.0)):
        tot = 0.0
        for x, wq in zip(xs, ws):
            for ra in ras:
                a, b = fo.antenna_ab(lat, gamma, lst, ra, math.asin(x))
                tot += wq * (a * a + b * b) / (2 * len(ras))
        assert abs(tot - golden["antenna_sky_average_a2_plus_b2"]) < 1e-12
    # a source on the rotation axis sees a time-independent a^2 + b^2
    vals = [sum(v * v for v in fo.antenna_ab(0.7, 1.1, lst, 0.4, math.pi / 2)) for lst in np.linspace(0, 6, 13)]
    assert np.ptp(vals) < 1e-13


def _antenna_tables(wl):
    """Per-SFT detector geometry of the synthetic two-detector network (inputs: workloads.antenna_geometry)."""
    return W.antenna_geometry(wl)


def test_sky_dependent_weights_sum_to_one_and_reduce_to_given_weights():
    """Eq. (5): the weights of every sky point sum to 1, so on a constant spectrogram P = c the statistic is c
    for every template; the weighted count of an all-hit spectrogram is 1; z is (s - 1)/sigma_G with
    sigma_G^2 = sum w^2 recomputed here from the antenna functions.  Catches: missing normalisation, weights
    taken at the wrong SFT / sky point, sigma_G from the wrong weights."""
    wl = W.config2(n_sft=96, n_sky=6, band_hz=0.05)
    wl.P[:] = np.float32(3.0)
    ant = _antenna_tables(wl)
    o = fo.Oracle(wl, antenna=ant)
    power, count, wcount, _, z, sigma = o.eval_range_z()
    assert np.allclose(power, 3.0, rtol=1e-12) and np.all(count == wl.n_sft) and np.allclose(wcount, 1.0, rtol=1e-12)
    g = wl.grid
    for i_sky in range(len(g.sky)):
        n = g.sky[i_sky]
        ra, dec = math.atan2(n[1], n[0]), math.asin(n[2])
        u = np.array([sum(v * v for v in fo.antenna_ab(ant[0][a], ant[1][a], ant[2][a], ra, dec)) for a in range(wl.n_sft)])
        w = u * wl.w.astype(np.float64)
        w /= w.sum()
        j = int(g.ravel(i_sky, 0, 0, 0, 0, 0))
        assert abs(sigma[j] - math.sqrt((w ** 2).sum())) < 1e-12 * sigma[j]
        assert abs(z[j] - (3.0 - 1.0) / sigma[j]) < 1e-8
    # weights vary across the sky (otherwise the feature is vacuous)
    assert np.ptp(sigma) > 1e-3 * sigma.mean()
    # an isotropic antenna factor (u = const) must give back the weights as given: emulate with P = hits only at one SFT
    wl2 = W.config2(n_sft=96, n_sky=6, band_hz=0.05)
    wl2.P[:] = 0.0
    wl2.P[17, :] = 1.0
    p2 = fo.Oracle(wl2, antenna=ant).eval_range()[0]
    n = g.sky[2]
    ra, dec = math.atan2(n[1], n[0]), math.asin(n[2])
    u = np.array([sum(v * v for v in fo.antenna_ab(ant[0][a], ant[1][a], ant[2][a], ra, dec)) for a in range(wl.n_sft)])
    w = u * wl2.w.astype(np.float64)
    assert abs(p2[int(g.ravel(2, 0, 0, 0, 0, 5))] - w[17] / w.sum()) < 1e-15


def test_standardised_statistic_is_zero_mean_unit_variance_in_noise(golden):
    """Eq. (36) with Eq. (13)-(14): z ~ N(0, 1) on an Exponential(1) spectrogram.  Catches: sigma_G from sum w
    instead of sum w^2, mu_G off by the chi^2 factor 2, z not using the template's own weights."""
    wl = W.config2(n_sft=400, n_sky=3)
    for ant in (None, _antenna_tables(wl)):
        o = fo.Oracle(wl, antenna=ant)
        n_f0 = wl.grid.n_f0
        power, _, _, _, z, sigma = o.eval_range_z(0, n_f0)
        assert abs(z.mean() - golden["z_noise_mean"]) < 4 / math.sqrt(n_f0)
        assert abs(z.var() - golden["z_noise_var"]) < 4 * math.sqrt(2.0 / n_f0) + 0.05
        if ant is None:   # fixed weights: mu_G = sum w, sigma_G = sqrt(sum w^2), recomputed here
            w = wl.w.astype(np.float64)
            assert np.allclose(z, (power - w.sum()) / math.sqrt((w ** 2).sum()), rtol=0, atol=1e-9)
            assert np.allclose(sigma, math.sqrt((w ** 2).sum()), rtol=1e-12)


def test_standardised_statistic_with_per_bin_weights_uses_row_means():
    """Eq. (36) under per-(SFT, bin) weights (reading R21): the box-level weights are the row means
    m_a = mean_k w[a][k] over the n_bins bins of the spectrogram, so sigma_G = sqrt(sum_a m_a^2) and
    z = (s - sum_a m_a) / sigma_G for EVERY template, recomputed here in numpy from the weight array alone.
    Catches: a mean over the leading dimension instead of n_bins, a missing division, the gathered w[a][k_a] used
    in the moments, sigma_G from sum m instead of sum m^2."""
    wl = W.config4(n_sft=120, n_sky=4, band_hz=0.2, n_lines=5)
    assert wl.per_bin_weights
    # the last two columns become row padding (ld = n_bins + 2): a mean over the leading dimension would differ
    nb = wl.n_bins - 2
    wl.w[:, nb:] *= np.float32(7.0)
    o = fo.Oracle(wl)
    o.pb.n_bins -= 2
    power, _, _, _, z, sigma = o.eval_range_z()
    m = wl.w[:, :nb].astype(np.float64).mean(axis=1)      # [n_sft] row means over the n_bins bins
    assert not np.allclose(m, wl.w.astype(np.float64).mean(axis=1), rtol=1e-6)
    mu, sg = m.sum(), math.sqrt((m ** 2).sum())
    assert np.allclose(sigma, sg, rtol=1e-12, atol=0) and np.ptp(sigma) == 0.0
    assert np.allclose(z, (power - mu) / sg, rtol=0, atol=1e-9)
    # the line bins make rows uneven: the gathered weight differs from the row mean, so a slip would show
    assert abs(power.mean() - mu) < 0.2 * mu and np.ptp(wl.w, axis=1).max() > 0.0
    # the statistic itself is the gathered-weight sum: brute force for three templates
    for idx in (0, int(power.size // 2), int(power.size - 1)):
        k, _, rc = o.track(idx)
        assert rc == 0
        a = np.arange(wl.n_sft)
        assert abs(power[idx] - (wl.w[a, k].astype(np.float64) * wl.P[a, k].astype(np.float64)).sum()) < 1e-12


# ---------------------------------------------------------------- boxes and the veto (:496-502)
def test_topk_per_region_against_python_sorted():
    """Catches: wrong region index, veto applied after instead of before the selection, tie order."""
    rng = np.random.Generator(np.random.PCG64(3))
    n_pt, n_f0, bpb, k = 12, 10, 4, 3
    vals = rng.integers(0, 6, n_pt * n_f0).astype(np.float64)      # many exact ties
    pbox = np.array([0, 0, 1, 1, 1, 2, 2, 0, 3, 3, 3, 3])
    keep = rng.random(n_pt * n_f0) < 0.7
    got = fo.topk_per_region(vals, n_f0, bpb, k, pbox=pbox, keep=keep)
    n_bands = 3
    assert len(got) == 4 * n_bands
    for r, (gi, gv) in enumerate(got):
        pb, band = divmod(r, n_bands)
        members = [(-(vals[i]), i) for i in range(vals.size)
                   if pbox[i // n_f0] == pb and (i % n_f0) // bpb == band and keep[i]]
        ref = sorted(members)[:k]
        assert [int(i) for i in gi] == [i for _, i in ref]
        assert list(gv) == [-v for v, _ in ref]
    # one box of points and no veto = the per-band top-k
    a = fo.topk_per_region(vals, n_f0, bpb, k)
    b = fo.topk_per_band(vals, n_f0, bpb, k)
    assert all(np.array_equal(x[0], y[0]) for x, y in zip(a, b))


def test_explicit_templates_z_equals_grid_z_and_bank_loudest_under_veto():
    """fto_eval_templates_z: a list that enumerates the grid gives eval_range_z's z and sigma_G exactly (fixed and
    sky-dependent weights, where sigma_G differs between sky points); loudest_of_bank against Python's sorted().
    Catches: z from another template's weights, the veto applied after the maximum, the tie order."""
    wl = W.config2(n_sft=96, n_sky=5, band_hz=0.05)
    g = wl.grid
    recs = [(g.f0_start + i * g.df0, g.f1_start + j * g.df1, s[0], s[1], s[2], 0.0, 86400.0, g.t_ref)
            for s in g.sky for j in range(g.n_f1) for i in range(g.n_f0)]
    tl = np.array(recs, dtype=fo.TEMPLATE_DTYPE)
    for ant in (None, W.antenna_geometry(wl)):
        o = fo.Oracle(wl, antenna=ant)
        a = o.eval_range_z()
        b = fo.eval_templates_z(o, tl, g.t_ref)
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        if ant is not None:
            assert np.ptp(b[5]) > 1e-3 * b[5].mean()
    power, _, wcount, _, z, _ = b
    floor = float(np.quantile(wcount, 0.7))
    for by_z in (False, True):
        key = z if by_z else power
        ref = sorted((-(key[i]), i) for i in range(key.size) if wcount[i] >= floor)[0][1]
        assert fo.loudest_of_bank(power, wcount, z, floor, by_z) == ref
    assert fo.loudest_of_bank(power, wcount, z, 2.0 * wcount.max()) == -1
    assert fo.loudest_of_bank([1.0, 3.0, 3.0], [1, 1, 1], [0, 0, 0]) == 1


def test_mismatch_definition_eq24():
    """Eq. (24): m = 0 at the matched template, m = 1 for a template that recovers only the noise mean."""
    assert fo.mismatch(3.0, 3.0, 1.0) == 0.0 and fo.mismatch(3.0, 1.0, 1.0) == 1.0
    assert abs(fo.mismatch(3.0, 2.5, 1.0) - 0.25) < 1e-15


def test_number_of_templates_eq_a10_against_quadrature_and_bank_density():
    """N(Delta lambda) (Eq. 29 with the density of Eq. A9, closed form Eq. A10) against (a) numerical quadrature of
    rho = k f0^5 a_p^2 Omega^3 over the box, one axis at a time (Simpson), and (b) the bank itself: a xi-uniform bank
    puts the fraction N(sub-box) / N(box) of its templates into a sub-box.  Catches: a wrong exponent or factor 1/(p+1),
    P_orb used where Omega is meant, a missing 2 pi of phi_b, sky as delta instead of sin delta."""
    from scipy.integrate import simpson
    box = dict(f0_lo=100.0, f0_hi=100.125, f1_lo=0.0, f1_hi=0.0, ra_lo=0.3, ra_hi=1.1, sd_lo=-0.2, sd_hi=0.5,
               ap_lo=2.0, ap_hi=7.0, porb_lo=12 * 86400.0, porb_hi=40 * 86400.0, t_ref=0.0)
    T_sft, T_obs, voc = 900.0, 180 * 86400.0, 1e-4
    k = T_sft ** 6 * T_obs * voc ** 2

    def quad(lo, hi, p):
        x = np.linspace(lo, hi, 20001)
        return simpson(x ** p, x=x)
    num = (k * quad(box["f0_lo"], box["f0_hi"], 5) * (box["ra_hi"] - box["ra_lo"]) * (box["sd_hi"] - box["sd_lo"])
           * quad(box["ap_lo"], box["ap_hi"], 2) * quad(2 * math.pi / box["porb_hi"], 2 * math.pi / box["porb_lo"], 3) * 2 * math.pi)
    N = fo.n_templates(box, T_sft, T_obs, voc)
    assert abs(N - num) < 1e-9 * num
    # k = T_SFT^6 T_obs (v/c)^2: N scales as the sixth power of T_SFT and linearly in T_obs
    assert abs(fo.n_templates(box, 2 * T_sft, 3 * T_obs, voc) / N - 64 * 3) < 1e-9
    # (b) the sub-box a_p < 5, P_orb < 20 d (i.e. Omega above 2 pi / 20 d), alpha < 0.6
    sub = dict(box, ap_hi=5.0, porb_hi=20 * 86400.0, ra_hi=0.6)
    frac = fo.n_templates(sub, T_sft, T_obs, voc) / N
    n = 200000
    tl = fo.bank_draw(box, 21, 0, n)
    ra = np.arctan2(tl["ny"], tl["nx"])
    inside = (tl["a_p"] < 5.0) & (tl["P_orb"] < 20 * 86400.0) & (ra < 0.6)
    assert abs(inside.mean() - frac) < 5 * math.sqrt(frac * (1 - frac) / n), (inside.mean(), frac)


def test_mismatch_sampler_noiseless_limits():
    """PAPER.md:320-324 on a NOISELESS spectrogram (P = 0 plus the signal), where the answer is known: s(lambda) =
    amp * sum w, mu_G = sum w, the best template recovers the fraction of SFTs on which its track coincides with the
    signal's, so m = 1 - (weighted fraction of coinciding SFTs) in [0, 1], recomputed here from the tracks alone; and
    a bank that contains the signal itself (zero-width box) gives m = 0 exactly.  Catches: the wrong sign or
    denominator of Eq. (24), the signal injected along another template's track, the maximum taken over the wrong bank."""
    wl = W.config3(n_sft=240, n_ap=2, n_porb=2, n_tasc=2, n_inj=0)
    wl.P[:] = 0.0
    g = wl.grid
    n = g.sky[0]
    ra = float(np.arctan2(n[1], n[0]) % (2 * math.pi)); sd = float(n[2])
    f_mid = g.f0_start + 0.5 * g.n_f0 * g.df0
    box = dict(f0_lo=f_mid, f0_hi=f_mid + 4 * g.df0, f1_lo=0.0, f1_hi=0.0, ra_lo=ra, ra_hi=ra + 1e-3, sd_lo=sd, sd_hi=sd + 1e-3,
               ap_lo=4.0, ap_hi=4.2, porb_lo=20 * 86400.0, porb_hi=20.5 * 86400.0, t_ref=g.t_ref)
    T_obs = float(wl.t_mid.max() - wl.t_mid.min())
    r = fo.mismatch_sampler(wl, box, n_inj=3, oversampling=0.0, seed=5, amp=2.0, T_obs=T_obs, n_bank=300)
    w = wl.w.astype(np.float64)
    o = fo.Oracle(wl)
    for j in range(3):
        sig = fo.bank_draw(box, 5, j, 1)
        ks, _, _ = o.track_template(sig[0], box["t_ref"])
        assert abs(r["s_signal"][j] - 2.0 * w.sum()) < 1e-12
        bank = fo.bank_draw(box, 5 + 1 + j, 0, 300)
        frac = np.array([w[(o.track_template(t, box["t_ref"])[0] == ks)].sum() for t in bank]) / w.sum()
        # mu_G = sum w enters Eq. (24) although the data hold no noise: m = (2 - 2 frac) / (2 - 1)
        assert abs(r["m"][j] - (2.0 - 2.0 * frac.max()) / (2.0 - 1.0)) < 1e-12
        assert int(r["best"][j]) == int(np.argmax(frac)) or np.sum(frac == frac.max()) > 1
    point = dict(box, f0_hi=box["f0_lo"], ra_hi=ra, sd_hi=sd, ap_hi=4.0, porb_hi=20 * 86400.0)
    # (phi_b still varies inside a zero-width box: pin the orbit phase by making the bank the signal's own stream)
    sig = fo.bank_draw(point, 9, 0, 1)
    wl2 = W.config3(n_sft=240, n_ap=2, n_porb=2, n_tasc=2, n_inj=0)
    wl2.P[:] = 0.0
    ks, _, _ = fo.Oracle(wl2).track_template(sig[0], g.t_ref)
    wl2.P[np.arange(wl2.n_sft), ks] += np.float32(2.0)
    sp = fo.eval_templates(fo.Oracle(wl2), sig, g.t_ref)[0]
    assert fo.mismatch(sp[0], sp[0], w.sum()) == 0.0


# ---------------------------------------------------------------- Eq. (A11): xi-uniform random banks
BOX = dict(f0_lo=100.0, f0_hi=200.0, f1_lo=-1e-9, f1_hi=0.0, ra_lo=0.0, ra_hi=2 * math.pi, sd_lo=-1.0, sd_hi=1.0,
           ap_lo=1.0, ap_hi=10.0, porb_lo=10 * 86400.0, porb_hi=60 * 86400.0, t_ref=1000.0)


def test_counter_generator_is_uniform_and_order_independent():
    """Catches: correlated coordinates, a stream that depends on the batch boundaries."""
    a = fo.bank_draw(BOX, 5, 0, 1000)
    b = np.concatenate([fo.bank_draw(BOX, 5, 0, 300), fo.bank_draw(BOX, 5, 300, 700)])
    assert a.tobytes() == b.tobytes()
    u = np.array([[fo.uniform(9, i, d) for d in range(7)] for i in range(20000)])
    assert np.all((u > 0) & (u < 1))
    assert np.all(np.abs(u.mean(axis=0) - 0.5) < 4 / math.sqrt(12 * 20000))
    assert np.all(np.abs(u.var(axis=0) - 1 / 12) < 0.003)
    assert np.all(np.abs(np.corrcoef(u.T) - np.eye(7)) < 0.04)
    assert np.all(np.abs(np.corrcoef(u[:-1, 0], u[1:, 0])[0, 1]) < 0.04)


def test_xi_bank_marginal_densities_follow_eq_a9(golden):
    """The marginals of a xi-uniform bank follow rho ∝ f0^5 a_p^2 Omega^3 (Eq. A9), uniform in (alpha, sin delta,
    phi_b).  The expected bin counts come from numerical quadrature of the density, not from the inverse map.
    Catches: a wrong exponent, Omega drawn as P_orb, phi_b not spanning one orbit, non-unit sky vectors."""
    n = 200000
    tl = fo.bank_draw(BOX, 11, 0, n)

    def check(x, lo, hi, p):
        edges = np.linspace(lo, hi, 9)
        got = np.histogram(x, edges)[0]
        grid = np.linspace(lo, hi, 8001)
        dens = grid ** p
        cum = np.concatenate([[0.0], np.cumsum(0.5 * (dens[1:] + dens[:-1]) * np.diff(grid))])
        exp = n * np.diff(np.interp(edges, grid, cum)) / cum[-1]
        assert np.all(np.abs(got - exp) < 5 * np.sqrt(exp) + 1), (p, got, exp)

    check(tl["f0"], BOX["f0_lo"], BOX["f0_hi"], golden["xi_exponent_f0"])
    check(tl["a_p"], BOX["ap_lo"], BOX["ap_hi"], golden["xi_exponent_ap"])
    Om = 2 * math.pi / tl["P_orb"]
    check(Om, 2 * math.pi / BOX["porb_hi"], 2 * math.pi / BOX["porb_lo"], golden["xi_exponent_omega"])
    check(np.mod(np.arctan2(tl["ny"], tl["nx"]), 2 * math.pi), 0.0, 2 * math.pi, 0)
    check(tl["nz"], -1.0, 1.0, 0)
    phi_b = (tl["t_asc"] - BOX["t_ref"]) * Om
    check(phi_b, 0.0, 2 * math.pi, 0)
    check(tl["f1"], BOX["f1_lo"], BOX["f1_hi"], 0)
    assert np.allclose(tl["nx"] ** 2 + tl["ny"] ** 2 + tl["nz"] ** 2, 1.0, atol=1e-14)
    # isolated bank: a_p = 0 exactly
    iso = dict(BOX, ap_lo=0.0, ap_hi=0.0)
    assert np.all(fo.bank_draw(iso, 11, 0, 100)["a_p"] == 0.0)


def test_xi_round_trip():
    """lambda -> xi (Eq. A11) -> lambda: the drawn template, pushed forward through xi = lambda^(p+1)/(p+1), lands
    at xi_min + u (xi_max - xi_min) with the generator's own u.  Catches: a wrong inverse map."""
    tl = fo.bank_draw(BOX, 3, 40, 50)
    for j, t in enumerate(tl):
        i = 40 + j
        for val, lo, hi, p1, d in ((t["f0"], BOX["f0_lo"], BOX["f0_hi"], 6, 0), (t["a_p"], BOX["ap_lo"], BOX["ap_hi"], 3, 3),
                                   (2 * math.pi / t["P_orb"], 2 * math.pi / BOX["porb_hi"], 2 * math.pi / BOX["porb_lo"], 4, 4)):
            xi, xl, xh = val ** p1 / p1, lo ** p1 / p1, hi ** p1 / p1
            assert abs((xi - xl) / (xh - xl) - fo.uniform(3, i, d)) < 1e-12
