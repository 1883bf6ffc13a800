"""Pins of the column-level wiring of the oracle (orc_column_fluxes / orc_iterate_re) that the ray-level pins do
not reach: the isothermal-layer grid, the per-column scales kscale and
f_star_scale (eq. 20), and the column-level warm start of the scattering sweeps through
orc_iterate_re's persisted upward fluxes.  CPU only."""
import dataclasses

import numpy as np
import pytest

from oracle import binding as orc
from paper_1606_05474_b200 import inputs

rep = dataclasses.replace


def par(inp, **kw):
    return rep(inp, params=dict(inp.params, **kw))


def rel(a, b):
    sc = np.maximum(np.abs(b[0]), np.abs(b[1]))
    return max(np.max(np.abs(a[0] - b[0]) / sc), np.max(np.abs(a[1] - b[1]) / sc))


# ---------------------------------------------------------------- isothermal-layer grid
def test_iso_grid_is_eq19_and_eq11_on_whole_layers():
    """isothermal_layers = 1 assembled here from the separately pinned pieces, following the paper's statement of
    the isothermal grid: n layers between n+1 interfaces, dtau_i = (P_i,inter - P_i+1,inter)/g *
    kappa_i with the layer's own (centre) P, T (eq. 19), one Planck value per layer (eq. 11,
    PAPER.md:143-149), fluxes at the interfaces, quadrature over g and bins (eq. 31-33).  A wrong pressure
    difference, a level stride of 2, interface instead of centre temperatures or a dropped weight fails."""
    inp = par(inputs.make_config(4, n_cols=2, n_bins=5, n_layers=9, n_g=3), isothermal_layers=1, n_scat=7)
    Fu, Fd = orc.fluxes(inp)
    p = inp.params
    n, nb, ng = p["n_layers"], p["n_bins"], p["n_g"]
    for c in range(2):
        up, dn = np.zeros(n + 1), np.zeros(n + 1)
        for l in range(nb):
            B = np.array([orc.planck_bin_mean(inp.bin_edges[l], inp.bin_edges[l + 1], inp.T0[c, i]) for i in range(n)])
            piB_int = np.pi * orc.planck_bin_mean(inp.bin_edges[l], inp.bin_edges[l + 1], inp.t_intern[c])
            for g in range(ng):
                kap = np.array([inp.kscale[c] * orc.kappa_interp(inp.ktab, inp.tab_log10p, inp.tab_t, inp.p_layer[i],
                                                                 inp.T0[c, i], l, g) for i in range(n)])
                dtau = (inp.p_interface[:-1] - inp.p_interface[1:]) / p["gravity"] * kap
                fu, fd = orc.ray_fluxes(dtau, B, B, inp.w0[l], inp.g0[l], p["D"], inp.f_star[l] * inp.f_star_scale[c],
                                        piB_int, 1 + p["n_scat"])
                w = inp.g_wts[g] * (inp.bin_edges[l + 1] - inp.bin_edges[l])
                up += w * fu
                dn += w * fd
        assert rel((Fu[c], Fd[c]), (up, dn)) < 1e-13


@pytest.mark.parametrize("n_scat,w0", [(0, 0.0), (-1, 0.6)])
def test_iso_grid_equals_sublayer_grid_for_isothermal_column_on_flat_table(n_scat, w0):
    """Splitting invariance of eq. 11: with B constant two sublayers act as one layer, so for an isothermal column
    on a table that is flat in (P, T) the interface fluxes of the two grids are identical -- exactly for w0 = 0 (one
    pass is exact) and for the coupled system's solution (direct solve) with scattering."""
    inp = inputs.make_config(1, n_bins=6, n_layers=12, n_g=2)
    flat = np.broadcast_to(inp.ktab[3:4, 5:6], inp.ktab.shape).copy()
    inp = rep(inp, ktab=flat, w0=np.full(6, w0), g0=np.full(6, 0.25 if w0 else 0.0), T0=np.full((1, 12), 900.0),
              t_intern=np.array([300.0]))
    a = orc.fluxes(par(inp, n_scat=n_scat, isothermal_layers=1))
    b = orc.fluxes(par(inp, n_scat=n_scat, isothermal_layers=0))
    assert rel(a, b) < 5e-13


def test_grids_converge_with_layer_count_non_isothermal_faster():
    """PAPER.md:191 'if a large enough number of isothermal layers is used, the isothermal and non-isothermal
    calculations should agree' and Fig. 9: the emergent flux of the isothermal grid approaches the
    non-isothermal reference as the layer count grows, while the non-isothermal grid is converged with far fewer layers."""
    def toa(n, iso):
        inp = par(inputs.make_config(2, n_bins=10, n_layers=n, n_g=2), isothermal_layers=iso, n_scat=-1)
        return orc.fluxes(inp)[0][0, -1]
    ref = toa(320, 0)
    e_iso = [abs(toa(n, 1) - ref) / ref for n in (20, 40, 80, 160)]
    e_non = [abs(toa(n, 0) - ref) / ref for n in (20, 40, 80)]
    assert e_iso[0] > e_iso[1] > e_iso[2] > e_iso[3]            # "the deviation decreases as the resolution increases"
    assert e_non[0] > e_non[1] > e_non[2]
    assert all(a < b for a, b in zip(e_non, e_iso))             # at equal layer count the non-isothermal grid is closer
    assert e_iso[0] > 3e-3 and e_iso[3] < 1e-4                  # and the two grids do agree in the limit (second order here)


# ---------------------------------------------------------------- per-column scales
def test_kscale_multiplies_the_table_and_f_star_scale_the_stellar_flux():
    """kscale = k is the same as a table multiplied by k, f_star_scale = s the same as f_star multiplied by s
    (eq. 20: F_dn at the top = f (R*/a)^2 pi B*, the per-column factor), with values != 1 that differ
    from column to column; and both matter."""
    inp = inputs.make_config(3, n_cols=3, n_bins=7, n_layers=10, n_g=3)
    inp = rep(inp, kscale=np.array([0.37, 1.0, 4.2]), f_star_scale=np.array([2.5e-3, 7.0e-2, 0.4]))
    Fu, Fd = orc.fluxes(inp)
    for c in range(3):
        one = inp.take_columns([c])
        scaled = rep(one, ktab=inp.ktab * inp.kscale[c], kscale=np.ones(1), f_star=inp.f_star * inp.f_star_scale[c],
                     f_star_scale=np.ones(1))
        assert rel((Fu[c:c + 1], Fd[c:c + 1]), orc.fluxes(scaled)) < 1e-13
        plain = rep(one, kscale=np.ones(1), f_star_scale=np.ones(1))
        assert c == 1 or rel((Fu[c:c + 1], Fd[c:c + 1]), orc.fluxes(plain)) > 1e-2
    # the RE iteration passes them on as well
    st = orc.iterate_re(inp, 4)
    c = 2
    one = inp.take_columns([c])
    scaled = rep(one, ktab=inp.ktab * inp.kscale[c], kscale=np.ones(1), f_star=inp.f_star * inp.f_star_scale[c],
                 f_star_scale=np.ones(1))
    assert np.max(np.abs(orc.iterate_re(scaled, 4)["T"][0] - st["T"][c])) < 1e-9


# ---------------------------------------------------------------- column-level warm start
def test_column_warm_start_continues_the_sweeps_across_evaluations():
    """'flux values are still known from the previous timestep'.  With the temperatures held fixed (a
    limiter of 1e-300 T makes every step vanish in fp64) two evaluations of 1 + 2 sweeps through orc_iterate_re's
    persisted upward fluxes are six sweeps: the persisted state equals that of ONE evaluation with n_scat = 5, and its
    quadrature over the interface levels is the bolometric F_up of a cold 6-sweep orc_fluxes call."""
    base = inputs.make_config(1, n_bins=9, n_layers=11, n_g=3)
    frozen = dict(dT_frac_max=1e-300, flux_floor=0.0)
    two = orc.iterate_re(par(base, warm_start=1, n_scat=2, **frozen), 2)
    one = orc.iterate_re(par(base, warm_start=1, n_scat=5, **frozen), 1)
    assert np.array_equal(two["T"], base.T0) and np.array_equal(one["T"], base.T0)
    assert np.array_equal(two["fup"], one["fup"])
    three = orc.iterate_re(par(base, warm_start=1, n_scat=2, **frozen), 1)
    assert not np.array_equal(three["fup"], one["fup"])                   # 3 sweeps are not 6
    Fu, _ = orc.fluxes(par(base, n_scat=5))
    dnu = np.diff(base.bin_edges)
    up = np.einsum("l,g,lgj->j", dnu, base.g_wts, two["fup"][0][:, :, ::2])
    assert np.max(np.abs(up - Fu[0]) / Fu[0]) < 1e-13
    # chained calls keep the state: 1 + 1 iterations == 2 iterations
    a = orc.iterate_re(par(base, warm_start=1, n_scat=2, **frozen), 1)
    b = orc.iterate_re(par(base, warm_start=1, n_scat=2, **frozen), 1, state=a)
    assert np.array_equal(b["fup"], two["fup"])
