"""Pins P4-P7, P10, P14 of the oracle: the two-stream sublayer
formulas and single-ray sweeps against closed forms, the ODE they solve, splitting invariance and
the exact E3 solution.  CPU only."""
import numpy as np
import pytest
from scipy import integrate, special

from oracle import binding as orc

PI = np.pi


def coeffs(dtau, w0, g0, D, B_lo, B_up, **kw):
    return orc.sublayer_coeffs(dtau, w0, g0, D, B_lo, B_up, **kw)


def step(dtau, w0, g0, D, B_lo, B_up, F_up_lo, F_dn_up, **kw):
    """One sublayer with both incoming fluxes given: returns (F_up at upper, F_dn at lower)."""
    c = coeffs(dtau, w0, g0, D, B_lo, B_up, **kw)
    if c.branch == 2:
        q = c.x * (F_up_lo - F_dn_up) / (2.0 + c.x)
        return F_up_lo - q, F_dn_up + q
    return ((c.xi * F_up_lo - c.beta * F_dn_up + c.S_up) / c.alpha,
            (c.xi * F_dn_up - c.beta * F_up_lo + c.S_dn) / c.alpha)


# ---------------------------------------------------------------- P4 Beer-Lambert
def test_P4_beer_lambert_pure_absorption():
    """w0 = 0, B = 0: F_dn(BOA) = F_top exp(-D sum dtau) (eq. 8-9)."""
    rng = np.random.default_rng(3)
    dtau = 10.0 ** rng.uniform(-6, 0.5, 40)
    z = np.zeros(40)
    for D in (2.0, 1.66):
        Fu, Fd = orc.ray_fluxes(dtau, z, z, 0.0, 0.0, D, 7.5, 0.0, 1)
        assert Fd[0] == pytest.approx(7.5 * np.exp(-D * dtau.sum()), rel=1e-13)
        assert Fd[-1] == 7.5
        # reflecting lower boundary with no internal flux (eq. 22 with T_intern = 0): F_up0 = F_dn0
        assert Fu[0] == Fd[0]
        assert Fu[-1] == pytest.approx(7.5 * np.exp(-2 * D * dtau.sum()), rel=1e-13)


# ---------------------------------------------------------------- P5 opaque isothermal
def test_P5_opaque_isothermal_column_emits_piB():
    """Isothermal, w0 = 0, optically thick: F_up(TOA) = 2 pi eps B = pi B for D = 2 (eq. 9)."""
    dtau = np.full(30, 5.0)
    B = np.full(30, 0.37)
    Fu, Fd = orc.ray_fluxes(dtau, B, B, 0.0, 0.0, 2.0, 0.0, 0.0, 1)
    assert Fu[-1] == pytest.approx(PI * 0.37, rel=1e-13)
    assert Fd[0] == pytest.approx(PI * 0.37, rel=1e-13)
    Fu, _ = orc.ray_fluxes(dtau, B, B, 0.0, 0.0, 1.66, 0.0, 0.0, 1)
    assert Fu[-1] == pytest.approx(2 * PI * 0.37 / 1.66, rel=1e-13)


# ---------------------------------------------------------------- P14 limits between the printed equations
def test_P14_eq15_reduces_to_eq10_eq11_eq9():
    D, eps = 2.0, 0.5
    B_lo, B_up, dt = 1.3, 0.9, 0.37
    F1u, F2d = 2.2, 0.4
    tr = np.exp(-D * dt)
    Bp = (B_lo - B_up) / dt
    # eq. 10 with G1 labelling: destination B first, source B times T
    up, dn = step(dt, 0.0, 0.0, D, B_lo, B_up, F1u, F2d)
    assert up == pytest.approx(tr * F1u + 2 * PI * eps * (B_up - tr * B_lo + eps * Bp * (1 - tr)), rel=1e-14)
    assert dn == pytest.approx(tr * F2d + 2 * PI * eps * (B_lo - tr * B_up - eps * Bp * (1 - tr)), rel=1e-14)
    # eq. 15 -> eq. 11 when B_lo = B_up, with eq. 12's v: beta - v == alpha + beta - xi (G5)
    w0, g0 = 0.6, 0.25
    c = coeffs(dt, w0, g0, D, 1.1, 1.1)
    r = np.sqrt((1 - w0) / (1 - w0 * g0))
    zp, zm = 0.5 * (1 + r), 0.5 * (1 - r)
    T = np.exp(-D * np.sqrt((1 - w0 * g0) * (1 - w0)) * dt)
    assert c.trans == pytest.approx(T, rel=1e-15)
    v = (zm ** 2 * T + zp ** 2) * (1 - T)
    beta = zp * zm * (1 - T ** 2)
    assert c.alpha == pytest.approx(zm ** 2 * T ** 2 - zp ** 2, rel=1e-14)
    assert c.beta == pytest.approx(beta, rel=1e-14)
    assert c.xi == pytest.approx((zm ** 2 - zp ** 2) * T, rel=1e-14)
    assert c.S_up == pytest.approx(2 * PI * eps * 1.1 * (beta - v), rel=1e-13)
    assert c.S_dn == pytest.approx(c.S_up, rel=1e-15)
    # eq. 11 -> eq. 9 at w0 = 0 (zeta+ = 1, zeta- = 0)
    up, dn = step(dt, 0.0, 0.0, D, 1.1, 1.1, F1u, F2d)
    assert up == pytest.approx(tr * F1u + 2 * PI * eps * 1.1 * (1 - tr), rel=1e-14)
    assert dn == pytest.approx(tr * F2d + 2 * PI * eps * 1.1 * (1 - tr), rel=1e-14)


def test_branches_and_thresholds():
    """PAPER.md:232 (dtau < 1e-4 -> isothermal prescription) and PAPER.md:212 (1 - w0 < 1e-6 -> eq. 14)."""
    assert coeffs(0.99e-4, 0.3, 0.0, 2.0, 1.0, 2.0).branch == 1
    assert coeffs(1.01e-4, 0.3, 0.0, 2.0, 1.0, 2.0).branch == 0
    assert coeffs(1.0, 1.0 - 0.5e-6, 0.0, 2.0, 1.0, 2.0).branch == 2
    assert coeffs(1.0, 1.0 - 2e-6, 0.0, 2.0, 1.0, 2.0).branch == 0
    # isothermal fallback uses the mean of the two end values (S2) and is continuous at the switch
    a = step(0.99999e-4, 0.3, 0.2, 2.0, 1.0, 1.02, 0.5, 0.25)
    b = step(1.00001e-4, 0.3, 0.2, 2.0, 1.0, 1.02, 0.5, 0.25)
    # jump is O(dtau^2) ~ 1e-8; using B_lo or B_up alone would jump by D dtau dB/2 ~ 2e-6
    assert abs(a[0] - b[0]) < 3e-8 and abs(a[1] - b[1]) < 3e-8
    # eq. 14 as printed
    up, dn = step(0.8, 1.0, 0.3, 2.0, 9.0, 9.0, 2.0, 0.5)
    x = 2.0 * (1 - 0.3) * 0.8
    assert up == pytest.approx(2.0 - x * (2.0 - 0.5) / (2 + x), rel=1e-15)
    assert dn == pytest.approx(0.5 + x * (2.0 - 0.5) / (2 + x), rel=1e-15)


# ---------------------------------------------------------------- P6 layer-splitting invariance
@pytest.mark.parametrize("w0,g0,D", [(0.0, 0.0, 2.0), (0.7, 0.3, 2.0), (0.4, -0.5, 1.66), (0.95, 0.6, 2.0)])
def test_P6_layer_splitting_invariance(w0, g0, D):
    """eq. 15 is the exact solution of the two-stream ODE for a source linear in tau, so splitting a
    sublayer in two (B interpolated linearly in tau) must leave every flux unchanged.  This fails
    for the printed B-subscripts (G1) and for eps/(1 + w0 g0) (G2)."""
    dtau = np.array([0.8, 0.05, 1.7, 0.3])
    B = np.array([2.0, 1.5, 1.4, 0.6, 0.2])          # levels 0..4 (0 = bottom)
    nsw = 400                                         # converged sweeps
    Fu, Fd = orc.ray_fluxes(dtau, B[:-1], B[1:], w0, g0, D, 1.3, 0.4, nsw)
    # split sublayer 2 at 30 % of its optical depth measured from its lower end
    f = 0.3
    Bmid = B[2] + f * (B[3] - B[2])
    dtau2 = np.array([0.8, 0.05, 1.7 * f, 1.7 * (1 - f), 0.3])
    B2 = np.array([2.0, 1.5, 1.4, Bmid, 0.6, 0.2])
    Fu2, Fd2 = orc.ray_fluxes(dtau2, B2[:-1], B2[1:], w0, g0, D, 1.3, 0.4, nsw)
    keep = [0, 1, 2, 4, 5]
    assert np.allclose(Fu2[keep], Fu, rtol=1e-12, atol=0)
    assert np.allclose(Fd2[keep], Fd, rtol=1e-12, atol=0)


# ---------------------------------------------------------------- P7 the ODE itself
def _two_stream_rhs(tau, F, w0, g0, D, Bfun):
    """Two-stream ODE in tau (increasing downward) of Heng et al. (2014) that eq. 8, 11, 13 and 14
    of the paper solve: dF_up/dtau = ga F_up - gs F_dn - gB B ; dF_dn/dtau = -ga F_dn + gs F_up + gB B."""
    ga = D * (1.0 - 0.5 * w0 * (1.0 + g0))
    gs = D * 0.5 * w0 * (1.0 - g0)
    gB = 2.0 * PI * (1.0 - w0)
    B = Bfun(tau)
    return [ga * F[0] - gs * F[1] - gB * B, -ga * F[1] + gs * F[0] + gB * B]


def _bvp(dtau, w0, g0, D, B_lo, B_up, F_up_lo, F_dn_up):
    """Brute force: F_dn given at tau = 0 (upper level), F_up given at tau = dtau (lower level).
    Linear problem: shoot twice and combine."""
    Bfun = lambda t: B_up + (B_lo - B_up) * t / dtau
    def shoot(fu0):
        sol = integrate.solve_ivp(_two_stream_rhs, (0.0, dtau), [fu0, F_dn_up], method="DOP853",
                                  args=(w0, g0, D, Bfun), rtol=1e-13, atol=1e-15)
        return sol.y[0, -1], sol.y[1, -1]
    a0, d0 = shoot(0.0)
    a1, d1 = shoot(1.0)
    fu0 = (F_up_lo - a0) / (a1 - a0)            # F_up(lower) is affine in F_up(upper)
    return fu0, d0 + fu0 * (d1 - d0)


@pytest.mark.parametrize("dtau,w0,g0,D,B_lo,B_up", [
    (0.9, 0.0, 0.0, 2.0, 1.0, 1.0),      # eq. 9  (printed, unambiguous)  -> pins the ODE
    (0.9, 0.6, 0.3, 2.0, 1.0, 1.0),      # eq. 11 (printed, unambiguous)  -> pins the ODE
    (0.4, 0.5, -0.5, 1.66, 0.7, 0.7),    # eq. 11, D != 2, back scattering
    (1.2, 0.0, 0.0, 2.0, 2.0, 0.5),      # eq. 10 / G1
    (0.7, 0.7, 0.3, 2.0, 2.0, 0.5),      # eq. 15 / G1 + G2
    (2.5, 0.3, -0.4, 1.66, 0.2, 1.9),    # inverted gradient, D != 2
    (0.05, 0.9, 0.6, 2.0, 1.0, 1.4),
])
def test_P7_sublayer_solves_two_stream_ode(dtau, w0, g0, D, B_lo, B_up):
    F_up_lo, F_dn_up = 1.7, 0.6
    up, dn = step(dtau, w0, g0, D, B_lo, B_up, F_up_lo, F_dn_up)
    up_ref, dn_ref = _bvp(dtau, w0, g0, D, B_lo, B_up, F_up_lo, F_dn_up)
    assert up == pytest.approx(up_ref, rel=2e-11)
    assert dn == pytest.approx(dn_ref, rel=2e-11)


def test_P7_ode_reproduces_eq14_at_w0_one():
    """The same ODE at w0 = 1 gives eq. 14, so the ODE is the paper's."""
    up, dn = step(0.8, 1.0, 0.3, 2.0, 0.0, 0.0, 2.0, 0.5)
    up_ref, dn_ref = _bvp(0.8, 1.0, 0.3, 2.0, 0.0, 0.0, 2.0, 0.5)
    assert up == pytest.approx(up_ref, rel=1e-11) and dn == pytest.approx(dn_ref, rel=1e-11)


def test_general_solution_approaches_eq14_near_w0_one():
    """continuity of the switch — just below the threshold eq. 11 ~ eq. 14."""
    a = step(0.8, 1.0 - 2e-6, 0.3, 2.0, 0.0, 0.0, 2.0, 0.5)
    b = step(0.8, 1.0, 0.3, 2.0, 0.0, 0.0, 2.0, 0.5)
    assert a[0] == pytest.approx(b[0], rel=1e-5) and a[1] == pytest.approx(b[1], rel=1e-5)


# ---------------------------------------------------------------- P10 exact solution, eq. 3-7
def test_P10_exact_transmissivity_and_diffusivity():
    """eq. 6: T = (1-dt)e^-dt + dt^2 E1(dt) = 2 E3(dt); eq. 7 against the stored values of
    tests/golden/diffusivity_eq7.txt (to 1e-6) for the oracle's closed form and its brute-force quadrature; Fig. 1
    limits."""
    L = orc.lib()
    for dt in (1e-3, 1e-2, 0.1, 1.0, 10.0):
        closed = (1 - dt) * np.exp(-dt) + dt * dt * special.exp1(dt)
        assert closed == pytest.approx(2 * special.expn(3, dt), rel=1e-12)
        assert L.orc_exact_transmissivity_quadrature(dt, 200000) == pytest.approx(closed, rel=1e-9)
    Dex = lambda dt: -np.log(2 * special.expn(3, dt)) / dt
    import os
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "diffusivity_eq7.txt"))
    for dt, D in gold:
        assert -np.log(L.orc_exact_transmissivity(dt)) / dt == pytest.approx(D, abs=2e-7)      # eq. 7 with the oracle's eq. 6
        assert -np.log(L.orc_exact_transmissivity_quadrature(dt, 200000)) / dt == pytest.approx(D, abs=2e-7 + 5e-9 / dt)
    assert Dex(1e-6) == pytest.approx(2.0, abs=1e-4) and 1.0 < Dex(300.0) < 1.03       # Fig. 1: 2 -> 1
    d = [Dex(x) for x in np.geomspace(1e-4, 50, 60)]
    assert np.all(np.diff(d) < 0)                 # monotone from 2 to 1


def test_P10_eq4_is_the_exact_formal_solution():
    """eq. 4 against brute-force angular integration of the formal solution of
    eq. 1 for a linear-in-tau source; fixes the labelling used for G1."""
    dt, B_lo, B_up, Fin_up, Fin_dn = 0.7, 2.0, 0.9, 1.1, 0.3
    Bp = (B_lo - B_up) / dt
    def inner(mu):          # emission reaching the top along mu; t = optical distance from the top
        f = lambda t: (B_up + Bp * t) * np.exp(-t / mu) / mu
        return integrate.quad(f, 0, dt, epsabs=0, epsrel=1e-13)[0]
    emis = integrate.quad(lambda mu: 2 * mu * inner(mu), 0, 1, epsabs=0, epsrel=1e-11)[0]
    trans = 2 * special.expn(3, dt)
    up_ref = trans * Fin_up + PI * emis
    up, dn = orc.exact_layer_eq4(dt, trans, B_lo, B_up, Fin_up, Fin_dn)
    assert up == pytest.approx(up_ref, rel=1e-10)
    def inner_dn(mu):       # t = optical distance from the bottom
        f = lambda t: (B_lo - Bp * t) * np.exp(-t / mu) / mu
        return integrate.quad(f, 0, dt, epsabs=0, epsrel=1e-13)[0]
    emis = integrate.quad(lambda mu: 2 * mu * inner_dn(mu), 0, 1, epsabs=0, epsrel=1e-11)[0]
    assert dn == pytest.approx(trans * Fin_dn + PI * emis, rel=1e-10)


def test_P10b_E1_and_closed_form_transmissivity():
    """O8c: E_1 against scipy.special.exp1 and eq. 6's closed form against 2 E_3, across the
    series / continued-fraction switch and from dtau = 1e-12 to 700."""
    L = orc.lib()
    xs = np.concatenate([np.geomspace(1e-12, 700.0, 400), [0.999999, 1.0, 1.000001, 2.0, 50.0]])
    for x in xs:
        assert L.orc_expint_E1(x) == pytest.approx(special.exp1(x), rel=2e-14, abs=1e-300)
        # absolute: T multiplies fluxes and 1 - T multiplies pi B, both of order one
        assert abs(L.orc_exact_transmissivity(x) - 2 * special.expn(3, x)) < 3e-15
    assert L.orc_exact_transmissivity(0.0) == 1.0


def test_P10b_exact_ray_is_the_layer_solution_chained_and_splits_exactly_for_isothermal_B():
    """O8c: (i) the ray routine is eq. 4 chained with eq. 20/22; (ii) eq. 3 is exact for an isothermal
    slab whatever the splitting ONLY through T = 2 E_3 of the whole slab for the emergent intensity
    moments -- not for fluxes (angular distribution changes), so instead: (iii) optically thick
    isothermal column => F_up(TOA) = pi B, F_dn(BOA) = pi B, and with B = 0 the transmitted flux is
    f_star * prod_s 2 E_3(dtau_s)."""
    rng = np.random.default_rng(3)
    N = 12
    dtau = 10.0 ** rng.uniform(-3, 0.7, N)
    B = np.sort(rng.uniform(0.2, 2.0, N + 1))[::-1].copy()
    Fu, Fd = orc.ray_fluxes_exact(dtau, B[:-1], B[1:], 1.3, 0.4)
    fd = 1.3
    for s in range(N - 1, -1, -1):
        _, fd = orc.exact_layer_eq4(dtau[s], 2 * special.expn(3, dtau[s]), B[s], B[s + 1], 0.0, fd)
        assert Fd[s] == pytest.approx(fd, rel=1e-13)
    fu = Fd[0] + 0.4
    assert Fu[0] == fu
    for s in range(N):
        fu, _ = orc.exact_layer_eq4(dtau[s], 2 * special.expn(3, dtau[s]), B[s], B[s + 1], fu, 0.0)
        assert Fu[s + 1] == pytest.approx(fu, rel=1e-13)
    thick = np.full(8, 30.0)
    Fu, Fd = orc.ray_fluxes_exact(thick, np.ones(8), np.ones(8), 0.0, 0.0)
    assert Fu[-1] == pytest.approx(PI, rel=1e-12) and Fd[0] == pytest.approx(PI, rel=1e-12)
    Fu, Fd = orc.ray_fluxes_exact(dtau, np.zeros(N), np.zeros(N), 2.0, 0.0)
    assert Fd[0] == pytest.approx(2.0 * np.prod(2 * special.expn(3, dtau)), rel=1e-12)


def test_P10_two_stream_D2_matches_exact_for_thin_layers():
    """north_star check (3): with D = 2 the two-stream single-layer result tends to the exact one
    (eq. 4 with eq. 6) as dtau -> 0, error O(dtau^2 ln dtau) relative to the emitted flux."""
    errs = []
    for dt in (1e-1, 1e-2, 1e-3):
        B_lo, B_up = 1.0, 0.8
        up, dn = step(dt, 0.0, 0.0, 2.0, B_lo, B_up, 0.5, 0.2, dtau_iso=0.0)
        upx, dnx = orc.exact_layer_eq4(dt, 2 * special.expn(3, dt), B_lo, B_up, 0.5, 0.2)
        errs.append(max(abs(up - upx), abs(dn - dnx)))
    assert errs[0] < 5e-2 and errs[1] < errs[0] / 20 and errs[2] < errs[1] / 20
    # and for an opaque layer both give pi B of the near side
    up, _ = step(80.0, 0.0, 0.0, 2.0, 1.0, 1.0, 0.5, 0.2)
    upx, _ = orc.exact_layer_eq4(80.0, 2 * special.expn(3, 80.0), 1.0, 1.0, 0.5, 0.2)
    assert up == pytest.approx(upx, rel=1e-12) and up == pytest.approx(PI, rel=1e-12)


# ---------------------------------------------------------------- conditioning of eq. 15 near dtau_iso
def test_eq15_source_loses_digits_for_nearly_conservative_layers_just_above_dtau_iso():
    """DESIGN.md section 4, limit (ii): for 1 - w0 ~ 1e-6 and dtau just above the 1e-4 switch the three
    terms of eq. 15 are of order r B ~ 1e-3 B and cancel to a source of order (1 - w0) D dtau B ~ 1e-12 B, and the B'
    term multiplies zeta_+ zeta_- (1 - T^2) -- itself good to 5e-10 only, since T is 1 to within 2e-7 -- by
    eps B'/(1 - w0 g0) ~ 5e3: evaluated in fp64 as printed the source of such a sublayer is off by tens of per cent OF
    ITSELF when the Planck function changes strongly across it (absolutely: < 1e-12 B, physically nil).  The oracle
    (plain fp64) against the same formulas in 60-digit decimal arithmetic on the same doubles."""
    from decimal import Decimal as Dc, getcontext
    getcontext().prec = 60

    def exact(dtau, w0, g0, D, B_lo, B_up):
        dtau, w0, g0, D, B_lo, B_up = (Dc(float(v)) for v in (dtau, w0, g0, D, B_lo, B_up))   # the doubles, exactly
        r = ((1 - w0) / (1 - w0 * g0)).sqrt()
        zp, zm = (1 + r) / 2, (1 - r) / 2
        tr = (-(D * ((1 - w0 * g0) * (1 - w0)).sqrt()) * dtau).exp()
        alpha, beta, xi = zm * zm * tr * tr - zp * zp, zp * zm * (1 - tr * tr), (zm * zm - zp * zp) * tr
        Bp, kp, eps = (B_lo - B_up) / dtau, 1 / (D * (1 - w0 * g0)), 1 / D
        pi = Dc("3.14159265358979323846264338327950288419716939937510582097494")
        S_up = 2 * pi * eps * (B_up * (alpha + beta) - B_lo * xi + kp * Bp * (alpha - xi - beta))
        return alpha, beta, xi, S_up

    def rel(a, b):
        return abs(float((Dc(float(a)) - b) / b))

    worst, worst_abs = {}, 0.0
    for name, w0, B_up in (("steep, nearly conservative", 1.0 - 1e-6, 1.0), ("flat, nearly conservative", 1.0 - 1e-6, 1.999),
                           ("steep, ordinary albedo", 0.5, 1.0)):
        errs = []
        for dtau in (1.3e-4, 2.7e-4, 5.1e-4, 9.9e-4):
            c = coeffs(dtau, w0, 0.3, 2.0, 2.0, B_up)
            a, b, x, s = exact(dtau, w0, 0.3, 2.0, 2.0, B_up)
            assert c.branch == 0
            assert rel(c.alpha, a) < 1e-12 and rel(c.xi, x) < 1e-12 and rel(c.beta, b) < 1e-8   # differences of O(1) terms
            errs.append(rel(c.S_up, s))
            worst_abs = max(worst_abs, abs(float(Dc(float(c.S_up)) - s)))
        worst[name] = max(errs)
    print("relative error of S_up, oracle vs 60 digits:", worst, "largest absolute error", worst_abs)
    assert 1e-3 < worst["steep, nearly conservative"] < 1.0         # measured 0.26: the digits are gone -- the method, in fp64
    assert worst["flat, nearly conservative"] < 1e-3                # measured 1.9e-4: the error scales with B_lo - B_up
    assert worst["steep, ordinary albedo"] < 1e-8                   # measured 2.9e-9
    assert worst_abs < 1e-11                                        # of B ~ 1: nil on the scale of any ordinary bin
