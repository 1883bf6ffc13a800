"""Pins P1, P2, P3, P11 of the oracle: Planck bin means, k-table
interpolation, column-mass closure, Gauss-Legendre quadrature.  CPU only."""
import ctypes as C
import numpy as np
import pytest
from scipy import integrate

from oracle import binding as orc
from paper_1606_05474_b200 import inputs

H, CL, KB = 6.62607015e-27, 2.99792458e10, 1.380649e-16


def planck_nu(nu, T):
    return 2.0 * H * CL * CL * nu ** 3 / np.expm1(H * CL * nu / (KB * T))


def test_sigma_sb_matches_codata():
    # CODATA 2018 value of the Stefan-Boltzmann constant in cgs (derived constant)
    assert orc.sigma_sb() == pytest.approx(5.670374419e-5, rel=1e-9)


@pytest.mark.parametrize("T", [60.0, 300.0, 1500.0, 6000.0])
def test_P1_bins_sum_to_sigma_T4_over_pi(T):
    """PAPER.md:253 (eq. 21): int pi B = sigma T^4.  Band covering x in [1e-3, 60]."""
    c2 = H * CL / KB
    edges = np.geomspace(1e-3, 60.0, 400) * T / c2
    tot = sum((edges[i + 1] - edges[i]) * orc.planck_bin_mean(edges[i], edges[i + 1], T)
              for i in range(edges.size - 1))
    # the part of the integral outside [1e-3, 60]: x^3/3 below (Rayleigh-Jeans), ~e^-60 x^3 above
    missing = (1e-3 ** 3 / 3.0 + np.exp(-60.0) * (60.0 ** 3 + 3 * 60.0 ** 2 + 6 * 60.0 + 6)) / (np.pi ** 4 / 15.0)
    assert tot * np.pi / (orc.sigma_sb() * T ** 4) == pytest.approx(1.0 - missing, abs=1e-12)


@pytest.mark.parametrize("T", [100.0, 777.0, 2900.0])
def test_P1_each_bin_vs_gauss_legendre(T):
    """Each bin mean against 64-point Gauss-Legendre of B_nu (the definition, O4)."""
    y, w = np.polynomial.legendre.leggauss(64)
    for edges in (np.linspace(500.0, 5000.0, 17), 1e4 / np.geomspace(30.0, 0.3, 301)[::15],
                  np.array([1.0, 5.0, 20.0, 60.0, 75.0])):   # last: x < 1 and straddling x = 1 at 100 K
        for lo, hi in zip(edges[:-1], edges[1:]):
            # split wide bins so the 64-point rule is converged
            sub = np.linspace(lo, hi, 9)
            ref = 0.0
            for a, b in zip(sub[:-1], sub[1:]):
                nu = 0.5 * (a + b) + 0.5 * (b - a) * y
                ref += 0.5 * (b - a) * np.sum(w * planck_nu(nu, T))
            ref /= (hi - lo)
            got = orc.planck_bin_mean(lo, hi, T)
            if ref > 1e-250:
                assert got == pytest.approx(ref, rel=2e-12)


def test_P1_series_agree_at_switch_and_total():
    """H(x) + G(x) = pi^4/15 for any x; both series must agree at the x = 1 switch."""
    L = orc.lib()
    for x in (0.05, 0.3, 0.999, 1.0):
        assert L.orc_planck_H_lower(x) + L.orc_planck_G_upper(x) == pytest.approx(np.pi ** 4 / 15, rel=3e-15)
    # library quadrature of the integrand as a third opinion
    val, _ = integrate.quad(lambda t: t ** 3 / np.expm1(t), 0.2, 0.9, epsabs=0, epsrel=1e-13)
    assert L.orc_planck_integral(0.2, 0.9) == pytest.approx(val, rel=1e-12)
    val, _ = integrate.quad(lambda t: t ** 3 / np.expm1(t), 0.7, 3.5, epsabs=0, epsrel=1e-13)
    assert L.orc_planck_integral(0.7, 3.5) == pytest.approx(val, rel=1e-12)


def test_planck_zero_temperature_is_zero():
    assert orc.planck_bin_mean(100.0, 200.0, 0.0) == 0.0     # PAPER.md:259 T_intern = 0


# ---------------------------------------------------------------- P2 opacity table
def _table():
    rng = np.random.default_rng(1)
    lp = np.linspace(0.0, 9.0, 7)
    tt = np.linspace(100.0, 2900.0, 15)
    k = rng.uniform(0.1, 10.0, (7, 15, 3, 2))
    return k, lp, tt


def test_P2_nodes_reproduced_exactly():
    k, lp, tt = _table()
    for ip in range(7):
        for it in range(15):
            assert orc.kappa_interp(k, lp, tt, 10.0 ** lp[ip], tt[it], 2, 1) == pytest.approx(k[ip, it, 2, 1], rel=1e-14)


def test_P2_exact_for_bilinear_table_and_linear_in_kappa_not_log():
    """'linearly interpolated across T and log P' (kappa itself, reading O3)."""
    _, lp, tt = _table()
    f = lambda x, t: 3.0 + 0.7 * x - 2e-3 * t + 1e-3 * x * t       # bilinear in (log10 P, T)
    k = f(lp[:, None], tt[None, :])[:, :, None, None] * np.ones((1, 1, 2, 2))
    rng = np.random.default_rng(2)
    for _ in range(50):
        x, t = rng.uniform(0.0, 9.0), rng.uniform(100.0, 2900.0)
        assert orc.kappa_interp(k, lp, tt, 10.0 ** x, t, 1, 0) == pytest.approx(f(x, t), rel=1e-13)
    # midpoint between two nodes in T: arithmetic (not geometric) mean
    k2, lp2, tt2 = _table()
    mid = orc.kappa_interp(k2, lp2, tt2, 10.0 ** lp2[3], 0.5 * (tt2[4] + tt2[5]), 0, 0)
    assert mid == pytest.approx(0.5 * (k2[3, 4, 0, 0] + k2[3, 5, 0, 0]), rel=1e-14)


def test_P2_clamps_outside_table():
    """PAPER.md:398 (fn. 9): outside the table -> closest tabulated value."""
    k, lp, tt = _table()
    assert orc.kappa_interp(k, lp, tt, 1e-5, 50.0, 0, 0) == pytest.approx(k[0, 0, 0, 0], rel=1e-14)
    assert orc.kappa_interp(k, lp, tt, 1e12, 5000.0, 1, 1) == pytest.approx(k[-1, -1, 1, 1], rel=1e-14)
    assert orc.kappa_interp(k, lp, tt, 10.0 ** lp[2], 5000.0, 1, 1) == pytest.approx(k[2, -1, 1, 1], rel=1e-14)
    # transposed-axis mistake would show here: P beyond range, T inside
    a = orc.kappa_interp(k, lp, tt, 1e12, tt[3], 1, 1)
    assert a == pytest.approx(k[-1, 3, 1, 1], rel=1e-14)


# ---------------------------------------------------------------- P3 column mass
def test_P3_constant_kappa_column_optical_depth():
    """eq. 19: sum of sublayer dtau = kappa (P_boa - P_toa)/g for constant kappa."""
    p_layer, p_int = inputs.pressure_grid(37, 1e9, 1.0)
    P = orc.level_pressures(p_layer, p_int)
    L = orc.lib()
    tot = sum(L.orc_sublayer_dtau(P[s], P[s + 1], 981.0, 0.3, 0.3) for s in range(P.size - 1))
    assert tot == pytest.approx(0.3 * (p_int[0] - p_int[-1]) / 981.0, rel=1e-13)
    # sublayer kappa is the mean of the two ends
    assert L.orc_sublayer_dtau(2000.0, 1000.0, 10.0, 1.0, 3.0) == pytest.approx(100.0 * 2.0)


def test_level_layout_and_interface_temperatures():
    """PAPER.md:230, Fig. 2: centres carry T; interfaces interpolated in log P (reading S1)."""
    p_layer, p_int = inputs.pressure_grid(6, 1e8, 1e2)
    P = orc.level_pressures(p_layer, p_int)
    assert np.all(np.diff(P) < 0) and P[0] == p_int[0] and P[-1] == p_int[-1] and P[1] == p_layer[0]
    # T linear in log P must be reproduced exactly at every level, ends included
    T = 900.0 + 55.0 * np.log(p_layer)
    Tl = orc.level_temperatures(p_layer, p_int, T)
    assert np.allclose(Tl, 900.0 + 55.0 * np.log(P), rtol=1e-13)
    # floor at 1 K on extrapolated ends
    Tl = orc.level_temperatures(p_layer, p_int, np.array([1.5, 300, 300, 300, 300, 300.0]))
    assert Tl[0] == 1.0


# ---------------------------------------------------------------- P11 quadrature
def test_P11_gauss_legendre_nodes_weights_eq32():
    """eq. 31-32: y_g roots of P_20, w_g = 2/((1-y^2) P'_20(y)^2)."""
    g, w = inputs.gauss_legendre_unit(20)
    y = 2.0 * g - 1.0
    P20 = np.polynomial.legendre.Legendre.basis(20)
    assert np.max(np.abs(P20(y))) < 1e-13
    w32 = 2.0 / ((1.0 - y ** 2) * P20.deriv()(y) ** 2)
    assert np.allclose(0.5 * w32, w, rtol=1e-12)
    assert np.sum(w) == pytest.approx(1.0, abs=1e-14)
    # exact for polynomials up to degree 39 on [0,1]
    assert np.sum(w * g ** 39) == pytest.approx(1.0 / 40.0, rel=1e-12)


def test_P11_constant_in_g_flux_is_returned_by_reduction():
    """If kappa does not depend on g, every g-ray carries the same flux, so the reduction must
    return the single-g result; and the bin sum must weight by the bin widths."""
    inp = inputs.make_config(0)
    k1 = inp.ktab[:, :, :, :1].copy()
    import dataclasses
    a = dataclasses.replace(inp, ktab=np.ascontiguousarray(np.repeat(k1, 4, axis=3)))
    b = dataclasses.replace(inp, ktab=np.ascontiguousarray(k1), g_pts=np.array([0.5]),
                            g_wts=np.array([1.0]), params=dict(inp.params, n_g=1))
    Fa, Da = orc.fluxes(a)
    Fb, Db = orc.fluxes(b)
    assert np.allclose(Fa, Fb, rtol=1e-13) and np.allclose(Da, Db, rtol=1e-13, atol=1e-300)
    # spectra x widths sum to the bolometric value
    Fu, Fd, su, sd = orc.fluxes(inp, want_spectra=True)
    dnu = np.diff(inp.bin_edges)
    assert np.sum(su[0] * dnu) == pytest.approx(Fu[0, -1], rel=1e-13)
    assert np.sum(sd[0] * dnu) == pytest.approx(Fd[0, 0], rel=1e-13)


# ---------------------------------------------------------------- O4b tabulated Planck function (reading S15)
def test_P16_tabulated_planck_nodes_linear_and_second_order():
    """PAPER.md:423 (Delta T = 10 K).  (i) at a node the table value is the bin mean itself; (ii) between two
    nodes the value is the straight line through them; (iii) the interpolation error falls like dT^2
    (ratio 25 between 50 K and 10 K) and is ~1e-4 relative at 10 K for a 1000 K level."""
    L = orc.lib()
    lo, hi = 2000.0, 2100.0
    assert L.orc_planck_bin_mean_tabulated(lo, hi, 1500.0, 10.0) == L.orc_planck_bin_mean(lo, hi, 1500.0)
    b0, b1 = L.orc_planck_bin_mean(lo, hi, 1230.0), L.orc_planck_bin_mean(lo, hi, 1240.0)
    assert L.orc_planck_bin_mean_tabulated(lo, hi, 1237.5, 10.0) == pytest.approx(b0 + 0.75 * (b1 - b0), rel=1e-14)
    ex = L.orc_planck_bin_mean(lo, hi, 1005.0)
    e10 = abs(L.orc_planck_bin_mean_tabulated(lo, hi, 1005.0, 10.0) - ex) / ex
    e50 = abs(L.orc_planck_bin_mean_tabulated(lo, hi, 1025.0, 50.0) - L.orc_planck_bin_mean(lo, hi, 1025.0)) / ex
    assert 1e-6 < e10 < 1e-4
    assert e50 / e10 == pytest.approx(25.0, rel=0.25)


def test_P16_tabulated_column_converges_to_exact_and_falls_back_above_the_table():
    import dataclasses
    inp = inputs.make_config(2, n_bins=30)
    ex = orc.fluxes(inp)
    sc = np.maximum(np.abs(ex[0]), np.abs(ex[1]))
    errs = []
    for dT in (50.0, 10.0, 2.0):
        t = orc.fluxes(dataclasses.replace(inp, params=dict(inp.params, planck_table_dT=dT, planck_table_Tmax=6000.0)))
        errs.append(np.max(np.abs(t[0] - ex[0]) / sc))
    assert errs[0] > errs[1] > errs[2] and errs[1] < 2e-4 and errs[2] < 1e-5
    assert errs[0] / errs[1] == pytest.approx(25.0, rel=0.4)
    # a column that reaches beyond the table uses the exact function throughout
    t = orc.fluxes(dataclasses.replace(inp, params=dict(inp.params, planck_table_dT=10.0, planck_table_Tmax=1500.0)))
    assert np.array_equal(t[0], ex[0]) and np.array_equal(t[1], ex[1])


# ---------------------------------------------------------------- P17 tabulated transmission function (S16)
def test_P17_tabulated_transmission_nodes_linear_in_log_kappa_and_error_bound():
    """O7b ("tabulate ... the transmission functions at ... a grid in ... opacity (Delta log10 kappa =
    0.1)"; reading S16).  (i) at a node the value is eq. 8 itself; (ii) between two nodes it is linear in log10 kappa;
    (iii) at the paper's step the absolute error stays below (dlog ln10)^2/8 * max|x(x-1)e^-x| = 2.1e-3 (the maximum, 0.309, is at x = 2.62) and is
    attained to within a factor 2; (iv) second order in the step."""
    L = orc.lib()
    c = 3.7
    for k in (-12, -3, 0, 5):
        kap = 10.0 ** (0.1 * k)
        assert L.orc_transmission_tabulated(c, kap, 0.1) == pytest.approx(np.exp(-c * kap), rel=1e-13)
    k0, k1 = 10.0 ** -0.3, 10.0 ** -0.2
    t0, t1 = np.exp(-c * k0), np.exp(-c * k1)
    for f in (0.25, 0.5, 0.9):
        kap = 10.0 ** (-0.3 + 0.1 * f)
        assert L.orc_transmission_tabulated(c, kap, 0.1) == pytest.approx(t0 + f * (t1 - t0), rel=1e-12)
    kap = np.geomspace(1e-4, 1e3, 4001)
    err = {}
    for dlog in (0.2, 0.1, 0.05):
        err[dlog] = max(abs(L.orc_transmission_tabulated(1.0, float(x), dlog) - np.exp(-x)) for x in kap)
    bound = lambda d: (d * np.log(10.0)) ** 2 / 8.0 * 0.309
    assert 0.5 * bound(0.1) < err[0.1] <= bound(0.1) * 1.02
    assert err[0.2] / err[0.1] == pytest.approx(4.0, rel=0.15) and err[0.1] / err[0.05] == pytest.approx(4.0, rel=0.1)
    assert L.orc_transmission_tabulated(1.0, 0.0, 0.1) == 1.0                      # no opacity: transparent


def test_P17_tabulated_transmission_column_error_report_and_limit():
    """Column level: the table changes the config-1-like fluxes by ~1e-4 at the paper's step (its error report), by
    several times less at half the step, and the step -> 0 limit is the exact run; opacities exactly on the nodes give
    the exact run; the Planck path and eq. 14 bins are untouched."""
    import dataclasses
    inp = inputs.make_config(1, n_bins=24, n_layers=30, n_g=4)
    ex = orc.fluxes(inp)
    sc = np.maximum(np.abs(ex[0]), np.abs(ex[1]))

    def dev(dlog, base=inp):
        r = orc.fluxes(dataclasses.replace(base, params=dict(base.params, trans_table_dlog10k=dlog)))
        return max(np.max(np.abs(r[0] - ex[0]) / sc), np.max(np.abs(r[1] - ex[1]) / sc))
    e1, e2, e3 = dev(0.1), dev(0.05), dev(1e-4)
    assert 1e-5 < e1 < 1e-2 and e2 < e1 / 3.0 and e3 < 1e-8
    # a table flat in (P, T) whose values sit on the nodes 10^(k/10): every sublayer's opacity is a node
    nodes = 10.0 ** (0.1 * np.round(10.0 * np.log10(inp.ktab[0, 0])))
    flat = dataclasses.replace(inp, ktab=np.broadcast_to(nodes, inp.ktab.shape).copy())
    a = orc.fluxes(flat)
    b = orc.fluxes(dataclasses.replace(flat, params=dict(flat.params, trans_table_dlog10k=0.1)))
    sa = np.maximum(np.abs(a[0]), np.abs(a[1]))
    assert max(np.max(np.abs(a[0] - b[0]) / sa), np.max(np.abs(a[1] - b[1]) / sa)) < 1e-11
    # pure-scattering bins (eq. 14) have no transmission function: a column of them does not change
    ps = dataclasses.replace(inp, w0=np.ones(24), params=dict(inp.params, n_scat=40))
    p0 = orc.fluxes(ps)
    p1 = orc.fluxes(dataclasses.replace(ps, params=dict(ps.params, trans_table_dlog10k=0.1)))
    assert np.array_equal(p0[0], p1[0]) and np.array_equal(p0[1], p1[1])
