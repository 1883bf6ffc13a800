"""Seeded synthetic inputs for the HELIOS two-stream hot path (BASELINE.json configs 0-4).

This module serves BOTH the CUDA path and the test oracle and therefore holds none of the
method's arithmetic (no interpolation, no two-stream coefficients, no sweeps, no reduction):
it only lays out grids, draws the random table / scattering / per-column parameters and
evaluates the *stellar model* (a blackbody, "The simplest approach is to adopt a
Planck function") by plain Gauss-Legendre quadrature so that the TOA boundary flux of eq. 20
 arrives at the C-ABI as an array, as SURVEY.md section 8(b) specifies.

Recipe: numpy default_rng(160605474 + cfg);
draw order a, b, phi, u (w0), g0, then per-column T0, T_irr, kscale.  All configs: gravity
1000 cm s^-2, D = 2, T_star = 6000 K, Gauss-Legendre g-points on [0,1].  The paper's real
k-tables, stellar spectra and planet data are not available offline; these arrays stand in for
them with the paper's shapes (101 layers 1 ubar-1 kbar, 300/3000 bins, 20 g, table step
200 K x 0.5 dex).
"""
from __future__ import annotations

import dataclasses
import numpy as np

SEED_BASE = 160605474
BAR = 1.0e6  # dyn cm^-2

# physical constants, cgs (CODATA 2018) -- used only for the stellar blackbody input
_H = 6.62607015e-27
_C = 2.99792458e10
_KB = 1.380649e-16


@dataclasses.dataclass
class HeliosInputs:
    """Everything one call sequence of the C-ABI needs, as float64/int32 numpy arrays."""
    name: str
    params: dict            # fields of helios_params (include/helios.h)
    p_layer: np.ndarray     # [n]    layer-centre P, index 0 = BOA
    p_interface: np.ndarray  # [n+1]
    bin_edges: np.ndarray   # [nb+1] cm^-1 ascending
    g_pts: np.ndarray       # [ng] on [0,1]
    g_wts: np.ndarray       # [ng] sum to 1
    ktab: np.ndarray        # [ntab_p][ntab_t][nb][ng] cm^2 g^-1
    tab_log10p: np.ndarray  # [ntab_p] log10(P / dyn cm^-2)
    tab_t: np.ndarray       # [ntab_t] K
    w0: np.ndarray          # [nb]
    g0: np.ndarray          # [nb]
    T0: np.ndarray          # [nc][n] start temperatures
    f_star: np.ndarray      # [nb] pi*B_l(T_star): TOA down-flux per unit wavenumber before scaling
    f_star_scale: np.ndarray  # [nc] (T_irr/T_star)^4  (= f (R_star/a)^2 of eq. 20)
    t_intern: np.ndarray    # [nc]
    kscale: np.ndarray      # [nc]
    run: dict               # what the config asks to run (max_iter, tol_dT, ...)
    kappa_scat: np.ndarray | None = None   # [nb] scattering opacity per bin, cm^2 g^-1 (helios_set_scattering), or None

    @property
    def n_cols(self) -> int:
        return int(self.T0.shape[0])

    def take_columns(self, idx) -> "HeliosInputs":
        """Sub-batch with the given column indices (columns are independent: SURVEY 8(e))."""
        idx = np.asarray(idx, dtype=np.int64)
        out = dataclasses.replace(
            self, T0=np.ascontiguousarray(self.T0[idx]),
            f_star_scale=np.ascontiguousarray(self.f_star_scale[idx]),
            t_intern=np.ascontiguousarray(self.t_intern[idx]),
            kscale=np.ascontiguousarray(self.kscale[idx]),
            params=dict(self.params, n_cols=int(idx.size)))
        return out


def gauss_legendre_unit(ng: int):
    """Gauss-Legendre nodes/weights mapped to [0,1] (eq. 31; weights sum to 1)."""
    y, w = np.polynomial.legendre.leggauss(ng)
    return 0.5 * (1.0 + y), 0.5 * w


def pressure_grid(n: int, p_boa: float, p_toa: float):
    """Centres log-spaced from p_boa (index 0) to p_toa; interfaces at half steps in log P."""
    if n == 1:
        q = p_toa / p_boa
        return np.array([p_boa * np.sqrt(q)]), np.array([p_boa, p_toa])
    q = (p_toa / p_boa) ** (1.0 / (n - 1))
    i = np.arange(n, dtype=np.float64)
    j = np.arange(n + 1, dtype=np.float64)
    return p_boa * q ** i, p_boa * q ** (j - 0.5)


def stellar_blackbody_bins(bin_edges: np.ndarray, t_star: float, npts: int = 96) -> np.ndarray:
    """pi * (bin mean of the Planck function at t_star), per unit wavenumber, by Gauss-Legendre
    quadrature inside each bin.  This is the *input* stellar model, not the method's Planck path."""
    y, w = np.polynomial.legendre.leggauss(npts)
    lo, hi = bin_edges[:-1, None], bin_edges[1:, None]
    nu = 0.5 * (lo + hi) + 0.5 * (hi - lo) * y[None, :]
    x = _H * _C * nu / (_KB * t_star)
    b = 2.0 * _H * _C * _C * nu ** 3 / np.expm1(x)
    return np.pi * 0.5 * np.sum(b * w[None, :], axis=1)


def synthetic_ktable(rng, ntab_p, ntab_t, nb, ng, g_pts):
    """k[iP][iT][l][g] = 10^(a_l + b_l y_g) (1 + 0.2 sin(2 pi iT/(nT-1) + phi_l) cos(pi iP/(nP-1)))."""
    a = rng.uniform(-4.0, 0.0, nb)
    b = rng.uniform(0.0, 4.0, nb)
    phi = rng.uniform(0.0, 2.0 * np.pi, nb)
    base = 10.0 ** (a[:, None] + b[:, None] * g_pts[None, :])            # [nb][ng]
    it = np.arange(ntab_t, dtype=np.float64) / max(ntab_t - 1, 1)
    ip = np.arange(ntab_p, dtype=np.float64) / max(ntab_p - 1, 1)
    mod = 1.0 + 0.2 * np.sin(2.0 * np.pi * it[None, :, None] + phi[None, None, :]) \
        * np.cos(np.pi * ip[:, None, None])                               # [nP][nT][nb]
    return np.ascontiguousarray(mod[:, :, :, None] * base[None, None, :, :])


def _default_params(nc, n, nb, ng, ntab_p, ntab_t, n_scat):
    return dict(n_cols=nc, n_layers=n, n_bins=nb, n_g=ng, ntab_p=ntab_p, ntab_t=ntab_t,
                precision=0, n_scat=n_scat, warm_start=0, isothermal_layers=0,
                D=2.0, gravity=1000.0, dtau_iso=1.0e-4, one_minus_w0_min=1.0e-6,
                dT_frac_max=0.1, T_floor=10.0, flux_floor=1.0e-7)


def make_config(cfg: int, n_cols: int | None = None, n_bins: int | None = None,
                n_layers: int | None = None, n_g: int | None = None) -> HeliosInputs:
    """Inputs of BASELINE.json config `cfg` (0..4).  The keyword overrides shrink a config for
    parity tests that the oracle must finish in seconds; the recipe is otherwise unchanged."""
    rng = np.random.default_rng(SEED_BASE + cfg)
    t_star = 6000.0
    if cfg == 0:
        nc, n, nb, ng = 1, 20, 16, 4
        ntab_p, ntab_t, t_lo, t_hi = 6, 6, 500.0, 2500.0
        p_boa, p_toa = 1.0e2 * BAR, 1.0e-4 * BAR
        n_scat = 0
    elif cfg in (1, 2, 3):
        nc, n, nb, ng = (1024 if cfg == 3 else 1), 100, 300, 20
        ntab_p, ntab_t, t_lo, t_hi = 20, 40, 100.0, 3000.0
        p_boa, p_toa = 1.0e3 * BAR, 1.0e-6 * BAR
        n_scat = 80 if cfg == 2 else 4
    elif cfg == 4:
        nc, n, nb, ng = 8192, 100, 1000, 20
        ntab_p, ntab_t, t_lo, t_hi = 20, 40, 100.0, 3000.0
        p_boa, p_toa = 1.0e3 * BAR, 1.0e-6 * BAR
        n_scat = 4
    else:
        raise ValueError("cfg must be 0..4")
    nc = n_cols if n_cols is not None else nc
    nb = n_bins if n_bins is not None else nb
    n = n_layers if n_layers is not None else n
    ng = n_g if n_g is not None else ng

    g_pts, g_wts = gauss_legendre_unit(ng)
    p_layer, p_interface = pressure_grid(n, p_boa, p_toa)
    if cfg == 0:
        bin_edges = np.linspace(500.0, 5000.0, nb + 1)
    else:  # log-spaced 0.3-30 um, converted to ascending wavenumber edges
        lam_um = np.geomspace(30.0, 0.3, nb + 1)
        bin_edges = 1.0e4 / lam_um
    tab_log10p = np.linspace(np.log10(p_toa), np.log10(p_boa), ntab_p)
    tab_t = np.linspace(t_lo, t_hi, ntab_t)
    ktab = synthetic_ktable(rng, ntab_p, ntab_t, nb, ng, g_pts)

    u = rng.uniform(0.0, 1.0, nb)
    g0_draw = rng.uniform(-0.3, 0.6, nb)
    if cfg == 0:
        w0 = np.zeros(nb)
        g0 = np.zeros(nb)
    elif cfg in (1, 2, 3):
        lam_c_um = 1.0e4 / (0.5 * (bin_edges[:-1] + bin_edges[1:]))
        w0 = 0.5 * u * np.minimum(1.0, (1.0 / lam_c_um) ** 4)   # Rayleigh-like lambda^-4, <= 0.5
        g0 = np.zeros(nb)
    else:
        w0 = 0.9 * u
        g0 = g0_draw

    if cfg == 0:
        T_start = np.full(nc, 1200.0)
        t_irr = np.zeros(nc)
        kscale = np.ones(nc)
        t_intern = np.full(nc, 100.0)
    elif cfg in (1, 2):
        T_start = np.full(nc, 1500.0)
        t_irr = np.full(nc, 1500.0)
        kscale = np.ones(nc)
        t_intern = np.zeros(nc)
    else:
        T_start = rng.uniform(800.0, 2200.0, nc)
        t_irr = rng.uniform(1000.0, 2500.0, nc)
        kscale = rng.uniform(0.5, 5.0, nc)
        t_intern = np.zeros(nc)
    T0 = np.repeat(T_start[:, None], n, axis=1)
    if cfg == 2:
        # one-shot evaluation on a fixed hot-Jupiter-like profile (stand-in for "cfg 1's converged
        # profile"): 1100 K aloft rising smoothly to 2300 K at depth
        lp = np.log10(p_layer / BAR)
        T0 = np.repeat((1100.0 + 1200.0 / (1.0 + np.exp(-(lp - 0.0) / 0.8)))[None, :], nc, axis=0)

    f_star = stellar_blackbody_bins(bin_edges, t_star)
    f_star_scale = (t_irr / t_star) ** 4

    run = {0: dict(flux_evals=1, re_iters=10, tol_dT=0.0, tol_flux=0.0),
           1: dict(flux_evals=0, re_iters=20000, tol_dT=1.0e-3, tol_flux=0.0),
           2: dict(flux_evals=1, re_iters=0, tol_dT=0.0, tol_flux=0.0),
           3: dict(flux_evals=0, re_iters=20000, tol_dT=1.0e-3, tol_flux=0.0),
           4: dict(flux_evals=0, re_iters=50, tol_dT=0.0, tol_flux=0.0)}[cfg]
    return HeliosInputs(
        name=f"config{cfg}", params=_default_params(nc, n, nb, ng, ntab_p, ntab_t, n_scat),
        p_layer=p_layer, p_interface=p_interface, bin_edges=np.ascontiguousarray(bin_edges),
        g_pts=g_pts, g_wts=g_wts, ktab=ktab, tab_log10p=tab_log10p, tab_t=tab_t,
        w0=np.ascontiguousarray(w0), g0=np.ascontiguousarray(g0),
        T0=np.ascontiguousarray(T0), f_star=f_star, f_star_scale=f_star_scale,
        t_intern=t_intern, kscale=kscale, run=run)


def shard_columns(n_cols: int, rank: int, world_size: int) -> range:
    """Contiguous, balanced column shard of `rank` (columns are independent, so multi-GPU is a
    pure partition with no data-path collective)."""
    base, rem = divmod(n_cols, world_size)
    start = rank * base + min(rank, rem)
    return range(start, start + base + (1 if rank < rem else 0))


M_PROTON_G = 1.67262192369e-24   # CODATA 2018


def rayleigh_h2_kappa(bin_edges: np.ndarray, mean_molecular_mass_g: float = 2.4 * M_PROTON_G) -> np.ndarray:
    """Input recipe for `kappa_scat`: the Rayleigh cross-section of molecular hydrogen, PAPER.md:193-206
    (eq. 16 with n_ref = 2.68678e19 cm^-3, K = 1 and the refractive index of eq. 17), evaluated at the centre
    wavenumber of every bin and divided by the mean molecular mass (sigma_scat / m-bar; PAPER.md:220:
    m-bar = 2.4 m_p for hydrogen-dominated atmospheres)."""
    nu = 0.5 * (np.asarray(bin_edges[:-1], dtype=np.float64) + np.asarray(bin_edges[1:], dtype=np.float64))
    lam = 1.0 / nu                                                     # cm
    n_ref = 2.68678e19
    n_lam = 13.58e-5 * (1.0 + 7.52e-11 / lam ** 2) + 1.0                # eq. 17
    sigma = 24.0 * np.pi ** 3 / (n_ref ** 2 * lam ** 4) * ((n_lam ** 2 - 1.0) / (n_lam ** 2 + 2.0)) ** 2   # eq. 16
    return sigma / mean_molecular_mass_g
