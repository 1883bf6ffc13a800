/*
 * helios_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the hot path of HELIOS (Malik et al.,
 * arXiv:1606.05474; text in /root/reference/PAPER.md, cited below as
 * "PAPER.md:<line>").  It follows the paper step by step in the paper's order
 * and notation, with the readings listed in DESIGN.md ("Readings of the
 * paper", items G1..G5 / S1..S15; S1..S10 are those of SURVEY.md section 8(c)).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code, header,
 * table or constant with paper_1606_05474_b200/csrc (the CUDA path), and the
 * CUDA path never calls it.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   orc_planck_*          P1  (sigma T^4/pi closure, Gauss-Legendre per bin)
 *   orc_kappa_interp      P2  (table nodes, bilinear exactness, clamping)
 *   orc_sublayer_dtau     P3  (column mass closure)
 *   orc_sublayer_coeffs /
 *   orc_ray_fluxes        P4 Beer-Lambert, P5 opaque isothermal pi*B,
 *                         P6 layer-splitting invariance, P7 ODE/BVP brute force,
 *                         P8 dense linear solve, P9 conservative scattering,
 *                         P10 exact E3 solution, P14 limits
 *   orc_column_fluxes     P11 quadrature
 *   orc_iterate_re        P12 fixed point (net flux = pi*sum(B_intern)),
 *                         P13 grey two-stream radiative equilibrium closed form.
 *   orc_ray_direct (O8b, n_sweeps <= 0; reading S12)
 *                         P8b numpy dense solve + the converged sweeps, P9 through it,
 *                         P8c closed form of the conservative column (exact rationals)
 *   orc_expint_E1, orc_exact_transmissivity, orc_ray_fluxes_exact (O8c; reading S13)
 *                         P10b scipy exp1 / 2 E_3, eq. 4 chained, opaque and B = 0 limits
 *   orc_ray_fluxes_w0s, kappa_scat in orc_column_fluxes (reading S14)
 *                         P15 dense solve with per-sublayer coefficients, flat-table
 *                         equivalence, zero opacity, eq. 16-17 by hand
 *   orc_planck_bin_mean_tabulated (O4b; reading S15)
 *                         P16 node exactness, linearity, second-order error, fall-back
 *   orc_transmission_tabulated, trans_table_dlog10k in orc_column_fluxes (O7b; reading S16)
 *                         P17 node exactness, linearity in log10 kappa, error bound 2.1e-3 and second order in the
 *                         step, column error report, step -> 0 limit
 *   orc_column_fluxes wiring (tests/test_oracle_wiring.py)
 *                         isothermal-layer grid: assembled from the pinned pieces following eq. 19 / eq. 11 on whole
 *                         layers; identical to the sublayer grid for an isothermal column on a flat table (splitting
 *                         invariance); the two grids converge with the layer count;
 *                         kscale == table x k and f_star_scale == f_star x s with values != 1;
 *                         column-level warm start: 2 x (1 + 2) sweeps through the persisted F_up == 6 cold sweeps
 *   eq. 7 / eq. 16-17     tests/golden/diffusivity_eq7.txt, rayleigh_h2.txt (scipy / 40-digit decimal arithmetic)
 *   PARITY UNPINNED (readings of a paper that is silent; only the fixed point and the limits are pinned): the
 *   *trajectory* of orc_iterate_re (limiter and oscillation rule S7, dead zone S11, order of updates), the
 *   interface-temperature rule (orc_level_temperatures: end-point extrapolation, S1) and the choice
 *   B_m = (B_lo+B_up)/2 in the isothermal fallback (S2).
 *
 * Units: cgs (P in dyn cm^-2, wavenumber in cm^-1, flux in erg s^-1 cm^-2).
 * Level numbering: n layers, levels 0..2n; even level 2j = interface j, odd level
 * 2i+1 = centre of layer i; level 0 = BOA, level 2n = TOA.
 * Sublayer s in [0,2n) lies between level s (lower) and level s+1 (upper).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* CODATA 2018 exact SI values in cgs. */
#define ORC_H  6.62607015e-27   /* erg s   */
#define ORC_C  2.99792458e10    /* cm s^-1 */
#define ORC_KB 1.380649e-16     /* erg K^-1 */
#define ORC_PI 3.14159265358979323846

typedef struct {
    int32_t n_layers, n_bins, n_g, ntab_p, ntab_t;
    int32_t n_scat;             /* extra sweeps after the first; -1 = direct solve (O8b) */
    int32_t warm_start;         /* 1: keep F_up between evaluations ("still known") */
    int32_t isothermal_layers;  /* 1: eq. 11 on whole layers */
    double D;                   /* diffusivity factor */
    double gravity;             /* cm s^-2, eq. 19 */
    double dtau_iso;            /* 1e-4 */
    double one_minus_w0_min;    /* 1e-6 */
    double dT_frac_max;         /* limiter, reading S7 */
    double T_floor;             /* limiter, reading S7 */
    double flux_floor;          /* dead zone, reading S11: a layer with |dF_i| < flux_floor * sigma T_i^4
                                   (eq. 29's own per-layer test) is left untouched */
    int32_t exact_absorption;   /* 1 = exact pure-absorption solution, eq. 3-6 (reading S13):
                                   w0, g0, D and n_scat are not used */
    double planck_table_dT;     /* > 0: Planck function of the levels from a table on the grid k * planck_table_dT
                                   (Delta T = 10 K), linear in T between the nodes (reading S15); 0 = exact */
    double planck_table_Tmax;   /* the table ends here; a column with a level at or above it uses the exact O4 */
    double trans_table_dlog10k; /* > 0: transmission function from a table on the opacity grid 10^(k * this) cm^2/g
                                   (Delta log10 kappa = 0.1), linear in log10 kappa between the nodes
                                   (reading S16); 0 = exact eq. 8 */
} orc_params;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* sigma_SB = 2 pi^5 k^4 / (15 h^3 c^2)  (eq. 21: integral of pi*B = sigma T^4). */
double orc_sigma_sb(void)
{
    const double pi5 = ORC_PI * ORC_PI * ORC_PI * ORC_PI * ORC_PI;
    const double k4 = ORC_KB * ORC_KB * ORC_KB * ORC_KB;
    return 2.0 * pi5 * k4 / (15.0 * ORC_H * ORC_H * ORC_H * ORC_C * ORC_C);
}

/* ------------------------------------------------------------------------- */
/* O4  Planck: bin-mean of B_nu~(T) = 2 h c^2 nu~^3 / (exp(h c nu~ / k T) - 1) */
/* ------------------------------------------------------------------------- */

/* Upper incomplete Planck integral G(x) = int_x^inf t^3/(e^t-1) dt
 *   = sum_{m>=1} e^{-m x} (x^3/m + 3x^2/m^2 + 6x/m^3 + 6/m^4)     (termwise integration
 * of t^3 e^{-mt}); used for x >= 1. */
double orc_planck_G_upper(double x)
{
    double sum = 0.0;
    for (int m = 1; m <= 400; ++m) {
        const double dm = (double)m;
        const double e = exp(-dm * x);
        const double term = e * (x * x * x / dm + 3.0 * x * x / (dm * dm)
                                 + 6.0 * x / (dm * dm * dm) + 6.0 / (dm * dm * dm * dm));
        sum += term;
        if (term <= 1e-18 * sum) break;
    }
    return sum;
}

/* Lower incomplete Planck integral H(x) = int_0^x t^3/(e^t-1) dt
 *   = sum_{k>=0} B_k x^{k+3} / (k! (k+3)),   t/(e^t-1) = sum_k B_k t^k/k!  (B_1 = -1/2);
 * used for x < 1 (radius of convergence 2 pi). */
double orc_planck_H_lower(double x)
{
    /* Bernoulli numbers B_0, B_1, B_2, B_4, ..., B_30 */
    static const double bern_even[] = {
        1.0 / 6.0, -1.0 / 30.0, 1.0 / 42.0, -1.0 / 30.0, 5.0 / 66.0, -691.0 / 2730.0,
        7.0 / 6.0, -3617.0 / 510.0, 43867.0 / 798.0, -174611.0 / 330.0, 854513.0 / 138.0,
        -236364091.0 / 2730.0, 8553103.0 / 6.0, -23749461029.0 / 870.0,
        8615841276005.0 / 14322.0 };
    double sum = x * x * x / 3.0;            /* k = 0: B_0 = 1, 0! = 1 */
    sum += -0.5 * x * x * x * x / 4.0;       /* k = 1: B_1 = -1/2, 1! = 1 */
    for (int j = 0; j < 15; ++j) {
        const int k = 2 * j + 2;             /* odd k > 1 have B_k = 0 */
        double fact = 1.0;                   /* k! */
        for (int q = 2; q <= k; ++q) fact *= (double)q;
        sum += bern_even[j] * pow(x, (double)(k + 3)) / (fact * (double)(k + 3));
    }
    return sum;
}

/* int_{x1}^{x2} t^3/(e^t-1) dt for 0 <= x1 <= x2, assembled so that no large constant
 * (pi^4/15) cancels: both below 1 -> H(x2)-H(x1); both above -> G(x1)-G(x2); straddling
 * -> [H(1)-H(x1)] + [G(1)-G(x2)]. */
double orc_planck_integral(double x1, double x2)
{
    if (x2 <= x1) return 0.0;
    if (x2 < 1.0) return orc_planck_H_lower(x2) - orc_planck_H_lower(x1);
    if (x1 >= 1.0) return orc_planck_G_upper(x1) - orc_planck_G_upper(x2);
    return (orc_planck_H_lower(1.0) - orc_planck_H_lower(x1))
         + (orc_planck_G_upper(1.0) - orc_planck_G_upper(x2));
}

/* Bin mean  B_l(T) = (1/dnu) int_{nu_lo}^{nu_hi} B_nu~(T) dnu~
 *                  = 2 k^4 T^4 / (h^3 c^2 dnu) * int_{x_lo}^{x_hi} t^3/(e^t-1) dt,  x = h c nu~/(k T).
 * erg s^-1 cm^-2 sr^-1 per cm^-1.  T <= 0 -> 0 (T_intern = 0). */
double orc_planck_bin_mean(double nu_lo, double nu_hi, double T)
{
    if (!(T > 0.0)) return 0.0;
    const double c2 = ORC_H * ORC_C / ORC_KB;   /* cm K */
    const double x_lo = c2 * nu_lo / T, x_hi = c2 * nu_hi / T;
    const double pref = 2.0 * ORC_KB * ORC_KB * ORC_KB * ORC_KB * T * T * T * T
                      / (ORC_H * ORC_H * ORC_H * ORC_C * ORC_C);
    return pref * orc_planck_integral(x_lo, x_hi) / (nu_hi - nu_lo);
}

/* ------------------------------------------------------------------------- */
/* O1/O2  staggered grid (Fig. 2 at 274)                  */
/* ------------------------------------------------------------------------- */

/* P_lev[2j] = p_interface[j], P_lev[2i+1] = p_layer[i]. */
void orc_level_pressures(int n, const double *p_layer, const double *p_interface, double *P_lev)
{
    for (int i = 0; i < n; ++i) { P_lev[2 * i] = p_interface[i]; P_lev[2 * i + 1] = p_layer[i]; }
    P_lev[2 * n] = p_interface[n];
}

/* Interface temperatures from centre temperatures, linear in log P (reading S1):
 * interior interface j between centres j-1 and j; the two end interfaces by linear
 * extrapolation in log P from the two nearest centres; floor at 1 K. */
void orc_level_temperatures(int n, const double *p_layer, const double *p_interface,
                            const double *T, double *T_lev)
{
    for (int i = 0; i < n; ++i) T_lev[2 * i + 1] = T[i];
    if (n == 1) { T_lev[0] = T[0]; T_lev[2] = T[0]; return; }
    for (int j = 0; j <= n; ++j) {
        int a = j - 1, b = j;                 /* centres below and above interface j */
        if (j == 0) { a = 0; b = 1; }
        if (j == n) { a = n - 2; b = n - 1; }
        const double la = log(p_layer[a]), lb = log(p_layer[b]), lj = log(p_interface[j]);
        const double w = (lj - la) / (lb - la);
        double t = T[a] + w * (T[b] - T[a]);
        if (t < 1.0) t = 1.0;
        T_lev[2 * j] = t;
    }
}

/* ------------------------------------------------------------------------- */
/* O3  opacity: bilinear in (log10 P, T), clamped (PAPER.md:376, 398 fn. 9)  */
/* ------------------------------------------------------------------------- */

/* ktab layout [ntab_p][ntab_t][n_bins][n_g]; axes uniform ascending. */
double orc_kappa_interp(const double *ktab, int ntab_p, int ntab_t, int n_bins, int n_g,
                        const double *tab_log10p, const double *tab_t,
                        double P, double T, int bin, int g)
{
    const double dlp = (tab_log10p[ntab_p - 1] - tab_log10p[0]) / (double)(ntab_p - 1);
    const double dt = (tab_t[ntab_t - 1] - tab_t[0]) / (double)(ntab_t - 1);
    double tp = (log10(P) - tab_log10p[0]) / dlp;
    if (tp < 0.0) tp = 0.0;
    if (tp > (double)(ntab_p - 1)) tp = (double)(ntab_p - 1);
    int ip = (int)floor(tp);
    if (ip > ntab_p - 2) ip = ntab_p - 2;
    const double fp = tp - (double)ip;
    double tt = (T - tab_t[0]) / dt;
    if (tt < 0.0) tt = 0.0;
    if (tt > (double)(ntab_t - 1)) tt = (double)(ntab_t - 1);
    int it = (int)floor(tt);
    if (it > ntab_t - 2) it = ntab_t - 2;
    const double ft = tt - (double)it;
    const size_t sp = (size_t)ntab_t * n_bins * n_g, st = (size_t)n_bins * n_g;
    const size_t o = (size_t)bin * n_g + g;
    const double k00 = ktab[ip * sp + it * st + o], k01 = ktab[ip * sp + (it + 1) * st + o];
    const double k10 = ktab[(ip + 1) * sp + it * st + o], k11 = ktab[(ip + 1) * sp + (it + 1) * st + o];
    return (1.0 - fp) * ((1.0 - ft) * k00 + ft * k01) + fp * ((1.0 - ft) * k10 + ft * k11);
}

/* O5  eq. 19 on a sublayer, kappa = mean of the two ends. */
double orc_sublayer_dtau(double P_lo, double P_up, double gravity, double kappa_lo, double kappa_up)
{
    return (P_lo - P_up) / gravity * 0.5 * (kappa_lo + kappa_up);
}

/* ------------------------------------------------------------------------- */
/* O6/O7  two-stream sublayer coefficients (eq. 8, 11-15)  */
/* ------------------------------------------------------------------------- */

typedef struct {
    int32_t branch;   /* 0 = non-isothermal eq. 15, 1 = isothermal eq. 11, 2 = pure scattering eq. 14 */
    int32_t pad_;
    double trans;     /* eq. 8 */
    double alpha, beta, xi;   /* eq. 12 */
    double S_up, S_dn;        /* bracketed source terms incl. the 2 pi eps factor */
    double x;                 /* D (1-g0) dtau of eq. 14 */
} orc_coeffs;

/*
 * One sublayer between a lower level (Planck B_lo, larger tau) and an upper level (B_up).
 * The fluxes then obey (eq. 11/15 with reading G1 for which B goes where and G2 for the
 * sign in eps/(1 - w0 g0)):
 *   F_up[upper] = (xi F_up[lower] - beta F_dn[upper] + S_up) / alpha
 *   F_dn[lower] = (xi F_dn[upper] - beta F_up[lower] + S_dn) / alpha
 * G1: the Planck value multiplying (alpha+beta) is the one at the level the flux arrives at
 *     (destination), the one multiplying xi is at the level it started from (source).  This is
 *     what the two-stream ODE gives; the printed eq. 15 carries the labels
 *     of Heng et al. (2014) where 1 is the upper interface.  Pinned by P6, P7, P10.
 * G2: the printed eps/(1 + w0 g0) is eps/(1 - w0 g0).  Pinned by P6, P7.
 * B' = dB/dtau with tau increasing downward = (B_lo - B_up)/dtau (eq. 5).
 */
/*
 * O7b  tabulated transmission function ("tabulate the Planck and the transmission functions at the
 * model's wavelength values and a grid in T (Delta T = 10 K) and opacity (Delta log10 kappa = 0.1)"; reading S16).
 * For one bin and one (sub)layer the transmission of eq. 8 is a function of the opacity alone,
 * T(kappa) = exp(-c kappa) with c = lambda * (column mass of the sublayer) = lambda dtau / kappa.  Nodes
 * kappa_k = 10^(k dlog), k integer; between two nodes the value is linear in log10 kappa.  (The nodes are evaluated
 * on the fly here, which gives the numbers a stored table would hold.)  kappa <= 0: T = 1.
 */
double orc_transmission_tabulated(double c, double kappa, double dlog)
{
    if (!(kappa > 0.0)) return 1.0;
    const double u = log10(kappa) / dlog;
    const double k = floor(u);
    const double f = u - k;
    const double t0 = exp(-c * pow(10.0, k * dlog));
    const double t1 = exp(-c * pow(10.0, (k + 1.0) * dlog));
    return t0 + f * (t1 - t0);
}

static void orc_sublayer_coeffs_core(double dtau, double w0, double g0, double D,
                                     double B_lo, double B_up, double dtau_iso, double one_minus_w0_min,
                                     double kappa_mean, double trans_dlog, orc_coeffs *c);

void orc_sublayer_coeffs(double dtau, double w0, double g0, double D,
                         double B_lo, double B_up, double dtau_iso, double one_minus_w0_min,
                         orc_coeffs *c)
{
    orc_sublayer_coeffs_core(dtau, w0, g0, D, B_lo, B_up, dtau_iso, one_minus_w0_min, 0.0, 0.0, c);
}

/* trans_dlog > 0: the transmission function comes from the table of O7b at the sublayer's opacity kappa_mean (the
 * kappa of eq. 19); everything else -- dtau in B' and in the dtau_iso test, eq. 14 -- is unchanged. */
static void orc_sublayer_coeffs_core(double dtau, double w0, double g0, double D,
                                     double B_lo, double B_up, double dtau_iso, double one_minus_w0_min,
                                     double kappa_mean, double trans_dlog, orc_coeffs *c)
{
    const double eps = 1.0 / D;                                        /* eq. 2 */
    memset(c, 0, sizeof *c);
    if ((1.0 - w0) < one_minus_w0_min) {
        c->branch = 2;
        c->x = D * (1.0 - g0) * dtau;                                  /* eq. 14 */
        c->trans = 1.0;
        return;
    }
    const double r = sqrt((1.0 - w0) / (1.0 - w0 * g0));
    const double zp = 0.5 * (1.0 + r), zm = 0.5 * (1.0 - r);           /* eq. 13 */
    const double lam = D * sqrt((1.0 - w0 * g0) * (1.0 - w0));
    const double tr = (trans_dlog > 0.0 && kappa_mean > 0.0)
                    ? orc_transmission_tabulated(lam * dtau / kappa_mean, kappa_mean, trans_dlog)   /* O7b */
                    : exp(-lam * dtau);                                /* eq. 8 */
    c->trans = tr;
    c->alpha = zm * zm * tr * tr - zp * zp;                            /* eq. 12 */
    c->beta = zp * zm * (1.0 - tr * tr);
    c->xi = (zm * zm - zp * zp) * tr;
    if (dtau < dtau_iso) {
        /* eq. 11 with beta - v == alpha + beta - xi (G5) and B = mean of the ends (S2) */
        const double Bm = 0.5 * (B_lo + B_up);
        c->branch = 1;
        c->S_up = 2.0 * ORC_PI * eps * Bm * (c->alpha + c->beta - c->xi);
        c->S_dn = c->S_up;
    } else {
        const double Bp = (B_lo - B_up) / dtau;                        /* eq. 5 */
        const double kp = eps / (1.0 - w0 * g0);                       /* G2 */
        c->branch = 0;
        c->S_up = 2.0 * ORC_PI * eps * (B_up * (c->alpha + c->beta) - B_lo * c->xi
                                        + kp * Bp * (c->alpha - c->xi - c->beta));
        c->S_dn = 2.0 * ORC_PI * eps * (B_lo * (c->alpha + c->beta) - B_up * c->xi
                                        + kp * Bp * (c->xi - c->alpha + c->beta));
    }
}

/* ------------------------------------------------------------------------- */
/* O8  sweeps for one ray                            */
/* ------------------------------------------------------------------------- */

/*
 * nsub sublayers, nsub+1 levels.  B_lo[s], B_up[s] are the Planck values at the two ends of
 * sublayer s (equal for the isothermal-layer grid).  F_dn[nsub] = F_dn_top (eq. 20).
 * n_sweeps = 1 + n_scat complete (down, BOA, up) passes.  warm = 0: the coupled up-fluxes
 * start as zero ("starting with the coupled dependencies as zero"); warm = 1:
 * F_up holds the previous evaluation's values on entry.
 * BOA (eq. 22): F_up[0] = F_dn[0] + piB_intern.
 */
static void orc_ray_direct(int nsub, const orc_coeffs *c, double F_dn_top, double piB_intern,
                           double *F_up, double *F_dn);

void orc_ray_fluxes_w0s(int nsub, const double *dtau, const double *B_lo, const double *B_up,
                        const double *w0s, double g0, double D, double dtau_iso, double one_minus_w0_min,
                        double F_dn_top, double piB_intern, int n_sweeps, int warm,
                        double *F_up, double *F_dn);

void orc_ray_fluxes(int nsub, const double *dtau, const double *B_lo, const double *B_up,
                    double w0, double g0, double D, double dtau_iso, double one_minus_w0_min,
                    double F_dn_top, double piB_intern, int n_sweeps, int warm,
                    double *F_up, double *F_dn)
{
    double *w0s = (double *)malloc(sizeof(double) * (size_t)(nsub > 0 ? nsub : 1));
    for (int s = 0; s < nsub; ++s) w0s[s] = w0;
    orc_ray_fluxes_w0s(nsub, dtau, B_lo, B_up, w0s, g0, D, dtau_iso, one_minus_w0_min, F_dn_top, piB_intern,
                       n_sweeps, warm, F_up, F_dn);
    free(w0s);
}

/* The same with a single-scattering albedo per sublayer ("functions of wavelength,
 * temperature and pressure", reading S14): w0s[s] enters the coefficients of
 * sublayer s, including the switch to eq. 14 "in this layer and waveband". */
void orc_ray_fluxes_tt(int nsub, const double *dtau, const double *kappa_mean, double trans_dlog,
                       const double *B_lo, const double *B_up,
                       const double *w0s, double g0, double D, double dtau_iso, double one_minus_w0_min,
                       double F_dn_top, double piB_intern, int n_sweeps, int warm,
                       double *F_up, double *F_dn);

void orc_ray_fluxes_w0s(int nsub, const double *dtau, const double *B_lo, const double *B_up,
                        const double *w0s, double g0, double D, double dtau_iso, double one_minus_w0_min,
                        double F_dn_top, double piB_intern, int n_sweeps, int warm,
                        double *F_up, double *F_dn)
{
    orc_ray_fluxes_tt(nsub, dtau, NULL, 0.0, B_lo, B_up, w0s, g0, D, dtau_iso, one_minus_w0_min, F_dn_top, piB_intern,
                      n_sweeps, warm, F_up, F_dn);
}

/* The same with the tabulated transmission function of O7b when trans_dlog > 0: kappa_mean[s] is the opacity of
 * sublayer s (the kappa of eq. 19). */
void orc_ray_fluxes_tt(int nsub, const double *dtau, const double *kappa_mean, double trans_dlog,
                       const double *B_lo, const double *B_up,
                       const double *w0s, double g0, double D, double dtau_iso, double one_minus_w0_min,
                       double F_dn_top, double piB_intern, int n_sweeps, int warm,
                       double *F_up, double *F_dn)
{
    orc_coeffs *c = (orc_coeffs *)malloc(sizeof(orc_coeffs) * (size_t)(nsub > 0 ? nsub : 1));
    for (int s = 0; s < nsub; ++s)
        orc_sublayer_coeffs_core(dtau[s], w0s[s], g0, D, B_lo[s], B_up[s], dtau_iso, one_minus_w0_min,
                                 kappa_mean ? kappa_mean[s] : 0.0, kappa_mean ? trans_dlog : 0.0, &c[s]);
    if (n_sweeps <= 0) {                               /* the coupled system itself */
        orc_ray_direct(nsub, c, F_dn_top, piB_intern, F_up, F_dn);
        free(c);
        return;
    }
    if (!warm) for (int s = 0; s <= nsub; ++s) F_up[s] = 0.0;
    F_dn[nsub] = F_dn_top;
    for (int sweep = 0; sweep < n_sweeps; ++sweep) {
        for (int s = nsub - 1; s >= 0; --s) {          /* down: level s+1 -> level s */
            if (c[s].branch == 2)
                F_dn[s] = F_dn[s + 1] + c[s].x * (F_up[s] - F_dn[s + 1]) / (2.0 + c[s].x);
            else
                F_dn[s] = (c[s].xi * F_dn[s + 1] - c[s].beta * F_up[s] + c[s].S_dn) / c[s].alpha;
        }
        F_up[0] = F_dn[0] + piB_intern;                /* eq. 22 */
        for (int s = 0; s < nsub; ++s) {               /* up: level s -> level s+1 */
            if (c[s].branch == 2)
                F_up[s + 1] = F_up[s] - c[s].x * (F_up[s] - F_dn[s + 1]) / (2.0 + c[s].x);
            else
                F_up[s + 1] = (c[s].xi * F_up[s] - c[s].beta * F_dn[s + 1] + c[s].S_up) / c[s].alpha;
        }
    }
    free(c);
}

/*
 * O8b  direct solve (n_scat = -1, reading S12).  The sweeps of
 * PAPER.md:292 are a block Gauss-Seidel iteration on one linear system: the two relations of every
 * sublayer (eq. 15, or eq. 14 for pure scattering) and the two boundary conditions (eq. 20, 22) in
 * the 2(nsub+1) unknowns F_dn[s], F_up[s].  "n_scat -> infinity" is the solution of that system;
 * here it is written out and solved by plain Gaussian elimination with partial pivoting.
 * Unknown x[2s] = F_dn[s], x[2s+1] = F_up[s].  Rows:
 *   0        :  F_up[0] - F_dn[0] = piB_intern                                        (eq. 22)
 *   2s+1     :  alpha F_dn[s]   - xi F_dn[s+1] + beta F_up[s]   = S_dn                (eq. 15, down)
 *   2s+2     :  alpha F_up[s+1] - xi F_up[s]   + beta F_dn[s+1] = S_up                (eq. 15, up)
 *   2nsub+1  :  F_dn[nsub] = F_dn_top                                                 (eq. 20)
 * (eq. 14 rows: (2+x) F_dn[s] - 2 F_dn[s+1] - x F_up[s] = 0, (2+x) F_up[s+1] - 2 F_up[s] - x F_dn[s+1] = 0.)
 * The matrix is stored dense; with this ordering every row has its entries within one column of
 * the diagonal, so the elimination loops skip the part that is structurally zero (pivoting can
 * bring up the next row only and widen a row to the right by one more column; BW = 4 is a margin).
 * Arithmetic: binary128.  The system's condition number grows like the column's scattering optical
 * depth (x_total of eq. 14 for w0 = 1); elimination in fp64 then loses kappa * 1e-16, e.g. 1e-10 at
 * x_total ~ 1e6, which the closed form of the conservative case shows (pin P8c:
 * F_dn[s] = F_dn_top + piB_intern * sum_{s' >= s} x_s'/2).  In binary128 that loss is ~1e-28.
 */
typedef __float128 orc_q;       /* gcc's IEEE binary128 (software arithmetic; +, -, *, / only) */

static void orc_ray_direct(int nsub, const orc_coeffs *c, double F_dn_top, double piB_intern,
                           double *F_up, double *F_dn)
{
    const int N = 2 * (nsub + 1);
    orc_q *A = (orc_q *)calloc((size_t)N * N, sizeof(orc_q));
    orc_q *rhs = (orc_q *)calloc((size_t)N, sizeof(orc_q));
#define ORC_A(i, j) A[(size_t)(i) * N + (j)]
#define ORC_QABS(v) ((v) < 0 ? -(v) : (v))
    ORC_A(0, 1) = 1.0; ORC_A(0, 0) = -1.0; rhs[0] = piB_intern;
    for (int s = 0; s < nsub; ++s) {
        const int rd = 2 * s + 1, ru = 2 * s + 2;
        const int dn_s = 2 * s, up_s = 2 * s + 1, dn_s1 = 2 * s + 2, up_s1 = 2 * s + 3;
        if (c[s].branch == 2) {
            ORC_A(rd, dn_s) = (orc_q)2.0 + c[s].x; ORC_A(rd, dn_s1) = -2.0; ORC_A(rd, up_s) = -c[s].x;
            ORC_A(ru, up_s1) = (orc_q)2.0 + c[s].x; ORC_A(ru, up_s) = -2.0; ORC_A(ru, dn_s1) = -c[s].x;
        } else {
            ORC_A(rd, dn_s) = c[s].alpha; ORC_A(rd, dn_s1) = -c[s].xi; ORC_A(rd, up_s) = c[s].beta;
            rhs[rd] = c[s].S_dn;
            ORC_A(ru, up_s1) = c[s].alpha; ORC_A(ru, up_s) = -c[s].xi; ORC_A(ru, dn_s1) = c[s].beta;
            rhs[ru] = c[s].S_up;
        }
    }
    ORC_A(N - 1, 2 * nsub) = 1.0; rhs[N - 1] = F_dn_top;
    const int BW = 4;                                   /* see the comment above */
    for (int k = 0; k < N; ++k) {
        const int ilast = (k + BW < N - 1) ? k + BW : N - 1, jlast = ilast;
        int piv = k;
        for (int i = k + 1; i <= ilast; ++i)
            if (ORC_QABS(ORC_A(i, k)) > ORC_QABS(ORC_A(piv, k))) piv = i;
        if (piv != k) {
            for (int j = k; j <= jlast; ++j) { const orc_q t = ORC_A(k, j); ORC_A(k, j) = ORC_A(piv, j); ORC_A(piv, j) = t; }
            const orc_q t = rhs[k]; rhs[k] = rhs[piv]; rhs[piv] = t;
        }
        for (int i = k + 1; i <= ilast; ++i) {
            if (ORC_A(i, k) == 0) continue;
            const orc_q f = ORC_A(i, k) / ORC_A(k, k);
            for (int j = k; j <= jlast; ++j) ORC_A(i, j) -= f * ORC_A(k, j);
            rhs[i] -= f * rhs[k];
        }
    }
    for (int k = N - 1; k >= 0; --k) {
        const int jlast = (k + BW < N - 1) ? k + BW : N - 1;
        orc_q v = rhs[k];
        for (int j = k + 1; j <= jlast; ++j) v -= ORC_A(k, j) * rhs[j];
        rhs[k] = v / ORC_A(k, k);
    }
#undef ORC_A
#undef ORC_QABS
    for (int s = 0; s <= nsub; ++s) { F_dn[s] = (double)rhs[2 * s]; F_up[s] = (double)rhs[2 * s + 1]; }
    free(A);
    free(rhs);
}

/*
 * O4b  tabulated Planck function ("tabulate the Planck ... functions at the model's wavelength
 * values and a grid in T (Delta T = 10 K)"; reading S15).  Nodes T_k = k dT, k = 0 ... ; the table value of a
 * bin at a node is the bin mean of O4; between nodes the value is linear in T.  (The nodes are evaluated on
 * the fly here, which gives the numbers a stored table would hold.)  The table ends at T_max; a column with
 * any level at or above T_max uses O4 throughout (decided by the caller).
 */
double orc_planck_bin_mean_tabulated(double nu_lo, double nu_hi, double T, double dT)
{
    const double t = T / dT;
    const int k = (int)t;
    const double f = t - (double)k;
    const double b0 = orc_planck_bin_mean(nu_lo, nu_hi, (double)k * dT);
    const double b1 = orc_planck_bin_mean(nu_lo, nu_hi, (double)(k + 1) * dT);
    return b0 + f * (b1 - b0);
}

/* ------------------------------------------------------------------------- */
/* O8c  exact solution in the pure-absorption limit        */
/* ------------------------------------------------------------------------- */

/*
 * Exponential integral E_1(x) = int_x^inf e^-t / t dt, x > 0 ("exponential integral of
 * the first order").  x <= 1: E_1 = -gamma - ln x - sum_{k>=1} (-x)^k / (k k!);  x > 1: the continued
 * fraction e^-x / (x + 1 - 1/(x + 3 - 4/(x + 5 - 9/(x + 7 - ...)))) evaluated by the modified Lentz
 * recurrence until two successive convergents agree to 1e-17.  Pinned against scipy.special.exp1.
 */
double orc_expint_E1(double x)
{
    const double euler_gamma = 0.57721566490153286060651209008240243;
    if (x <= 1.0) {
        double sum = 0.0, term = 1.0;                   /* term = (-x)^k / k! */
        for (int k = 1; k <= 60; ++k) {
            term *= -x / (double)k;
            const double add = -term / (double)k;
            sum += add;
            if (fabs(add) <= 1e-18 * fabs(sum)) break;
        }
        return -euler_gamma - log(x) + sum;
    }
    const double tiny = 1e-300;
    double b = x + 1.0, c = 1.0 / tiny, d = 1.0 / b, h = d;
    for (int i = 1; i <= 10000; ++i) {
        const double an = -(double)i * (double)i;
        b += 2.0;
        d = 1.0 / (an * d + b);
        c = b + an / c;
        const double del = c * d;
        h *= del;
        if (fabs(del - 1.0) <= 1e-17) break;
    }
    return h * exp(-x);
}

/* eq. 6: T = (1 - dtau) e^-dtau + dtau^2 E_1(dtau);  T(0) = 1. */
double orc_exact_transmissivity(double dtau)
{
    if (!(dtau > 0.0)) return 1.0;
    return (1.0 - dtau) * exp(-dtau) + dtau * dtau * orc_expint_E1(dtau);
}

/*
 * One ray in the pure-absorption limit: no coupling between the directions, one pass.
 * Sublayers with dtau >= dtau_iso: eq. 4 (orc_exact_layer_eq4 below; pinned by P10 against the
 * angular integration of the formal solution); thinner ones: eq. 3 with B = mean of the two ends
 * (reading S2, as for the two-stream formulas; it also avoids 0/0 in B' for dtau = 0).
 * BOA condition eq. 22, TOA condition eq. 20.
 */
void orc_exact_layer_eq4(double dtau, double trans, double B_lo, double B_up,
                         double F_up_lo, double F_dn_up, double *F_up_up, double *F_dn_lo);

void orc_ray_fluxes_exact(int nsub, const double *dtau, const double *B_lo, const double *B_up,
                          double dtau_iso, double F_dn_top, double piB_intern,
                          double *F_up, double *F_dn)
{
    double *tr = (double *)malloc(sizeof(double) * (size_t)(nsub > 0 ? nsub : 1));
    for (int s = 0; s < nsub; ++s) tr[s] = orc_exact_transmissivity(dtau[s]);
    double dummy;
    F_dn[nsub] = F_dn_top;                                               /* eq. 20 */
    for (int s = nsub - 1; s >= 0; --s) {
        if (dtau[s] < dtau_iso)
            F_dn[s] = tr[s] * F_dn[s + 1] + ORC_PI * 0.5 * (B_lo[s] + B_up[s]) * (1.0 - tr[s]);   /* eq. 3 */
        else
            orc_exact_layer_eq4(dtau[s], tr[s], B_lo[s], B_up[s], 0.0, F_dn[s + 1], &dummy, &F_dn[s]);
    }
    F_up[0] = F_dn[0] + piB_intern;                                      /* eq. 22 */
    for (int s = 0; s < nsub; ++s) {
        if (dtau[s] < dtau_iso)
            F_up[s + 1] = tr[s] * F_up[s] + ORC_PI * 0.5 * (B_lo[s] + B_up[s]) * (1.0 - tr[s]);   /* eq. 3 */
        else
            orc_exact_layer_eq4(dtau[s], tr[s], B_lo[s], B_up[s], F_up[s], 0.0, &F_up[s + 1], &dummy);
    }
    free(tr);
}

/* ------------------------------------------------------------------------- */
/* O9  one column: all rays + Gauss-weight x bin-width reduction             */
/* ------------------------------------------------------------------------- */

/* Neumaier-compensated accumulation: (sum, comp) += v */
static void orc_csum_add(double *sum, double *comp, double v)
{
    const double t = *sum + v;
    if (fabs(*sum) >= fabs(v)) *comp += (*sum - t) + v; else *comp += (v - t) + *sum;
    *sum = t;
}

/*
 * Bolometric interface fluxes of one column:
 *   F_up[j] = sum_l dnu_l sum_g w_g F_up(level of interface j; l, g),  same for F_dn.
 * g_wts are the weights on [0,1] (they sum to 1; the 1/2 of eq. 31 folded in, reading G4).
 * T[n]: layer-centre temperatures.  f_star[nb]: TOA downward flux per unit wavenumber (eq. 20),
 * multiplied by f_star_scale.  t_intern: eq. 21-22.  kscale multiplies every table value.
 * spec_up_toa / spec_dn_boa [nb]: sum_g w_g F at TOA (up) / BOA (down) per bin, or NULL.
 * fup_state: NULL, or [nb][ng][nsub+1] persisted up-fluxes for warm_start = 1.
 * inner_parallel: OpenMP over bins inside this call.
 * kappa_scat [nb] or NULL (reading S14): a scattering opacity per bin [cm^2/g], e.g. the
 *   Rayleigh cross-section of eq. 16-17 divided by the mean molecular mass.  It is added to the table
 *   (absorption) opacity at every level -- "its inclusion ... to the opacity of each model layer" -- and
 *   sets the single-scattering albedo of every sublayer, w0_s = kappa_scat / kappa_tot,s with kappa_tot,s
 *   the mean of the sublayer's two end values (the same mean as in eq. 19); w0[] is then not used,
 *   g0[] still is.  kscale multiplies the table value only.
 */
void orc_column_fluxes(const orc_params *p,
                       const double *p_layer, const double *p_interface, const double *bin_edges,
                       const double *g_wts, const double *ktab,
                       const double *tab_log10p, const double *tab_t,
                       const double *w0, const double *g0, const double *kappa_scat,
                       const double *T, const double *f_star, double f_star_scale,
                       double t_intern, double kscale,
                       double *F_up, double *F_dn, double *spec_up_toa, double *spec_dn_boa,
                       double *fup_state, int inner_parallel)
{
    const int n = p->n_layers, nb = p->n_bins, ng = p->n_g;
    const int iso = p->isothermal_layers;
    const int nsub = iso ? n : 2 * n, nlev = nsub + 1;
    const int lev_stride = iso ? 1 : 2;           /* level index of interface j = j*lev_stride */
    double *P_lev = (double *)malloc(sizeof(double) * (2 * n + 1));
    double *T_lev = (double *)malloc(sizeof(double) * (2 * n + 1));
    orc_level_pressures(n, p_layer, p_interface, P_lev);
    orc_level_temperatures(n, p_layer, p_interface, T, T_lev);

    /* S15: the Planck table spans 0 ... planck_table_Tmax */
    int use_ptab = p->planck_table_dT > 0.0;
    if (iso) {                                   /* the levels this grid evaluates B at */
        for (int i = 0; i < n && use_ptab; ++i)
            if (!(T[i] < p->planck_table_Tmax)) use_ptab = 0;
    } else {
        for (int v = 0; v <= 2 * n && use_ptab; ++v)
            if (!(T_lev[v] < p->planck_table_Tmax)) use_ptab = 0;
    }

    int any_scat = 0;
    for (int l = 0; l < nb; ++l) if (kappa_scat ? kappa_scat[l] > 0.0 : w0[l] > 0.0) any_scat = 1;
    /* w0 = 0 => beta = 0 => one sweep exact; n_scat = -1: direct solve of the coupled system (O8b) */
    const int n_sweeps = any_scat ? (p->n_scat < 0 ? 0 : 1 + p->n_scat) : 1;

    /* per-bin sums over g, reduced over bins afterwards in bin order (deterministic) */
    double *bin_up = (double *)malloc(sizeof(double) * (size_t)nb * (n + 1));
    double *bin_dn = (double *)malloc(sizeof(double) * (size_t)nb * (n + 1));

#pragma omp parallel for schedule(dynamic, 1) if (inner_parallel)
    for (int l = 0; l < nb; ++l) {
        double *dtau = (double *)malloc(sizeof(double) * nsub);
        double *B_lo = (double *)malloc(sizeof(double) * nsub);
        double *B_up = (double *)malloc(sizeof(double) * nsub);
        double *fu = (double *)malloc(sizeof(double) * nlev);
        double *fd = (double *)malloc(sizeof(double) * nlev);
        double *kap = (double *)malloc(sizeof(double) * (2 * n + 1));
        double *w0s = (double *)malloc(sizeof(double) * nsub);
        double *kbar = (double *)malloc(sizeof(double) * nsub);      /* the kappa of eq. 19 per sublayer (O7b) */
        const double ksc = kappa_scat ? kappa_scat[l] : 0.0;
        const double nu_lo = bin_edges[l], nu_hi = bin_edges[l + 1];
        /* O4: Planck at the levels this grid uses */
#define ORC_B_LEVEL(Tx) (use_ptab ? orc_planck_bin_mean_tabulated(nu_lo, nu_hi, (Tx), p->planck_table_dT) \
                                  : orc_planck_bin_mean(nu_lo, nu_hi, (Tx)))
        if (iso) {
            for (int i = 0; i < n; ++i)
                B_lo[i] = B_up[i] = ORC_B_LEVEL(T[i]);
        } else {
            double Bprev = ORC_B_LEVEL(T_lev[0]);
            for (int s = 0; s < nsub; ++s) {
                const double Bnext = ORC_B_LEVEL(T_lev[s + 1]);
                B_lo[s] = Bprev; B_up[s] = Bnext; Bprev = Bnext;
            }
        }
#undef ORC_B_LEVEL
        const double piB_int = ORC_PI * orc_planck_bin_mean(nu_lo, nu_hi, t_intern);
        for (int j = 0; j <= n; ++j) { bin_up[(size_t)l * (n + 1) + j] = 0.0; bin_dn[(size_t)l * (n + 1) + j] = 0.0; }
        for (int g = 0; g < ng; ++g) {
            /* O3 + O5 */
            if (iso) {
                for (int i = 0; i < n; ++i) {
                    const double k = kscale * orc_kappa_interp(ktab, p->ntab_p, p->ntab_t, nb, ng,
                                                               tab_log10p, tab_t, p_layer[i], T[i], l, g) + ksc;
                    dtau[i] = (p_interface[i] - p_interface[i + 1]) / p->gravity * k;   /* eq. 19 */
                    kbar[i] = k;
                    w0s[i] = kappa_scat ? ksc / k : w0[l];
                }
            } else {
                for (int v = 0; v <= 2 * n; ++v)
                    kap[v] = kscale * orc_kappa_interp(ktab, p->ntab_p, p->ntab_t, nb, ng,
                                                       tab_log10p, tab_t, P_lev[v], T_lev[v], l, g) + ksc;
                for (int s = 0; s < nsub; ++s) {
                    dtau[s] = orc_sublayer_dtau(P_lev[s], P_lev[s + 1], p->gravity, kap[s], kap[s + 1]);
                    kbar[s] = 0.5 * (kap[s] + kap[s + 1]);
                    w0s[s] = kappa_scat ? ksc / (0.5 * (kap[s] + kap[s + 1])) : w0[l];
                }
            }
            double *fu_use = fu;
            if (p->warm_start && fup_state) fu_use = fup_state + ((size_t)l * ng + g) * nlev;
            if (p->exact_absorption)
                orc_ray_fluxes_exact(nsub, dtau, B_lo, B_up, p->dtau_iso, f_star[l] * f_star_scale, piB_int,
                                     fu_use, fd);
            else
                orc_ray_fluxes_tt(nsub, dtau, kbar, p->trans_table_dlog10k, B_lo, B_up, w0s, g0[l], p->D, p->dtau_iso,
                                  p->one_minus_w0_min, f_star[l] * f_star_scale, piB_int, n_sweeps,
                                  (p->warm_start && fup_state) ? 1 : 0, fu_use, fd);
            for (int j = 0; j <= n; ++j) {
                bin_up[(size_t)l * (n + 1) + j] += g_wts[g] * fu_use[j * lev_stride];
                bin_dn[(size_t)l * (n + 1) + j] += g_wts[g] * fd[j * lev_stride];
            }
        }
        if (spec_up_toa) spec_up_toa[l] = bin_up[(size_t)l * (n + 1) + n];
        if (spec_dn_boa) spec_dn_boa[l] = bin_dn[(size_t)l * (n + 1) + 0];
        free(dtau); free(B_lo); free(B_up); free(fu); free(fd); free(kap); free(w0s); free(kbar);
    }

    for (int j = 0; j <= n; ++j) {
        double su = 0.0, cu = 0.0, sd = 0.0, cd = 0.0;
        for (int l = 0; l < nb; ++l) {
            const double dnu = bin_edges[l + 1] - bin_edges[l];
            orc_csum_add(&su, &cu, dnu * bin_up[(size_t)l * (n + 1) + j]);
            orc_csum_add(&sd, &cd, dnu * bin_dn[(size_t)l * (n + 1) + j]);
        }
        F_up[j] = su + cu;
        F_dn[j] = sd + cd;
    }
    free(P_lev); free(T_lev); free(bin_up); free(bin_dn);
}

/* nc independent columns (no exchange between columns). */
void orc_fluxes_batch(const orc_params *p, int nc,
                      const double *p_layer, const double *p_interface, const double *bin_edges,
                      const double *g_wts, const double *ktab,
                      const double *tab_log10p, const double *tab_t,
                      const double *w0, const double *g0, const double *kappa_scat /*[nb] or NULL*/,
                      const double *T /*[nc][n]*/, const double *f_star /*[nb]*/,
                      const double *f_star_scale /*[nc] or NULL*/, const double *t_intern /*[nc]*/,
                      const double *kscale /*[nc] or NULL*/,
                      double *F_up /*[nc][n+1]*/, double *F_dn /*[nc][n+1]*/,
                      double *spec_up_toa /*[nc][nb] or NULL*/, double *spec_dn_boa /*[nc][nb] or NULL*/)
{
    const int n = p->n_layers, nb = p->n_bins;
    const int outer = nc >= orc_num_threads();
#pragma omp parallel for schedule(dynamic, 1) if (outer)
    for (int c = 0; c < nc; ++c)
        orc_column_fluxes(p, p_layer, p_interface, bin_edges, g_wts, ktab, tab_log10p, tab_t, w0, g0, kappa_scat,
                          T + (size_t)c * n, f_star, f_star_scale ? f_star_scale[c] : 1.0,
                          t_intern[c], kscale ? kscale[c] : 1.0,
                          F_up + (size_t)c * (n + 1), F_dn + (size_t)c * (n + 1),
                          spec_up_toa ? spec_up_toa + (size_t)c * nb : NULL,
                          spec_dn_boa ? spec_dn_boa + (size_t)c * nb : NULL, NULL, !outer);
}

/* ------------------------------------------------------------------------- */
/* O10  radiative-equilibrium iteration (eq. 23-29)        */
/* ------------------------------------------------------------------------- */

/*
 * Sign history of one layer, packed in an int32 (the same packing is documented in
 * include/helios.h; each side implements it on its own):
 *   bits 0..11  six 2-bit codes, newest in bits 0..1; 0 = zero step, 1 = dT > 0, 2 = dT < 0
 *   bits 12..15 number of entries pushed so far, saturating at 6
 */
static int32_t orc_hist_push(int32_t h, double dT)
{
    const int32_t code = dT > 0.0 ? 1 : (dT < 0.0 ? 2 : 0);
    int32_t cnt = (h >> 12) & 0xF;
    if (cnt < 6) cnt++;
    return (cnt << 12) | (((h & 0xFFF) << 2) & 0xFFF) | code;
}

/* PAPER.md:309-311 with reading S7: returns the factor multiplying the layer's timestep
 * pre-factor: 0.67 if the last 6 steps strictly alternate in sign ("reduced by 33%"),
 * 1.1 if all 6 have the same non-zero sign ("increased by 10%"), else 1. */
static double orc_hist_factor(int32_t h)
{
    if (((h >> 12) & 0xF) < 6) return 1.0;
    int s[6];
    for (int k = 0; k < 6; ++k) s[k] = (h >> (2 * k)) & 3;
    int alternating = 1, monotone = (s[0] != 0);
    for (int k = 0; k < 5; ++k) {
        if (!((s[k] == 1 && s[k + 1] == 2) || (s[k] == 2 && s[k + 1] == 1))) alternating = 0;
        if (s[k + 1] != s[0]) monotone = 0;
    }
    if (alternating) return 0.67;
    if (monotone) return 1.1;
    return 1.0;
}

/*
 * Temperature step of layer i from the bolometric net fluxes (eq. 23-28 collapsed, reading S6;
 * sign per reading G3):
 *   dF_i = Fnet[i+1] - Fnet[i],  Fnet = F_up - F_dn                                  (eq. 23)
 *   dT_i = dF/(rho c_p dz) * f_pre * t_rad  with rho dz = dP/g, t_rad = c_p P/(sigma g T^3)
 *          (eq. 27), f_pre = 1e5/|dF|^0.9 (eq. 28)  =>  c_p, g, rho, dz cancel:
 *   dT_i = - a_i * 1e5 * (P_i/dP_i) * sgn(dF)|dF|^0.1 / (sigma T_i^3)
 *   the minus sign: energy conservation rho c_p dT/dt = -dFnet/dz with z upward (G3; eq. 24 as
 *   printed at PAPER.md:278 has no sign).  Then the limiter |dT| <= dT_frac_max * T (S7).
 */
double orc_re_delta_T(double dF, double a, double P_layer, double dP, double T,
                      double dT_frac_max)
{
    const double sigma = orc_sigma_sb();
    double dT = 0.0;
    if (dF != 0.0) {
        const double mag = pow(fabs(dF), 0.1);
        dT = -a * 1.0e5 * (P_layer / dP) * (dF > 0.0 ? mag : -mag) / (sigma * T * T * T);
    }
    const double lim = dT_frac_max * T;
    if (dT > lim) dT = lim;
    if (dT < -lim) dT = -lim;
    return dT;
}

/*
 * Iterate nc columns.  Per column and iteration, in this order (O10):
 *   fluxes(T) -> dT_i -> convergence test -> (if not converged) T_i <- max(T_i + dT_i, T_floor)
 *   -> push sgn(dT_i) -> a_i *= factor(history).
 * A column is converged when max_i |dT_i| < tol_dT (if tol_dT > 0) or
 * max_i |dF_i|/(sigma T_i^4) < tol_flux (eq. 29, if tol_flux > 0); a converged column is frozen
 * with the temperatures its last flux evaluation used.  iters[c] = number of flux evaluations.
 * step_factor (a_i, starts at 1) and sign_hist are in/out so that calls can be chained.
 * dT_last [nc][n] (or NULL): the last computed dT_i.  fup_state: see orc_column_fluxes.
 */
void orc_iterate_re(const orc_params *p, int nc,
                    const double *p_layer, const double *p_interface, const double *bin_edges,
                    const double *g_wts, const double *ktab,
                    const double *tab_log10p, const double *tab_t,
                    const double *w0, const double *g0, const double *kappa_scat /*[nb] or NULL*/,
                    double *T /*[nc][n] in/out*/, const double *f_star,
                    const double *f_star_scale, const double *t_intern, const double *kscale,
                    int max_iter, double tol_dT, double tol_flux,
                    double *step_factor /*[nc][n]*/, int32_t *sign_hist /*[nc][n]*/,
                    int32_t *iters /*[nc]*/, int32_t *converged /*[nc]*/,
                    double *dT_last, double *fup_state /*[nc][nb][ng][nlev] or NULL*/)
{
    const int n = p->n_layers, nb = p->n_bins, ng = p->n_g;
    const int nlev = (p->isothermal_layers ? n : 2 * n) + 1;
    const double sigma = orc_sigma_sb();
    const int outer = nc >= orc_num_threads();
#pragma omp parallel for schedule(dynamic, 1) if (outer)
    for (int c = 0; c < nc; ++c) {
        double *Tc = T + (size_t)c * n;
        double *a = step_factor + (size_t)c * n;
        int32_t *h = sign_hist + (size_t)c * n;
        double *Fu = (double *)malloc(sizeof(double) * (n + 1));
        double *Fd = (double *)malloc(sizeof(double) * (n + 1));
        double *dT = (double *)malloc(sizeof(double) * n);
        double *fs = fup_state ? fup_state + (size_t)c * nb * ng * nlev : NULL;
        if (converged[c]) { free(Fu); free(Fd); free(dT); continue; }   /* frozen by an earlier call */
        int it = 0, conv = 0;
        while (it < max_iter && !conv) {
            orc_column_fluxes(p, p_layer, p_interface, bin_edges, g_wts, ktab, tab_log10p, tab_t,
                              w0, g0, kappa_scat, Tc, f_star, f_star_scale ? f_star_scale[c] : 1.0,
                              t_intern[c], kscale ? kscale[c] : 1.0, Fu, Fd, NULL, NULL, fs, !outer);
            ++it;
            double max_dT = 0.0, max_rel = 0.0;
            for (int i = 0; i < n; ++i) {
                double dF = (Fu[i + 1] - Fd[i + 1]) - (Fu[i] - Fd[i]);                /* eq. 23 */
                /* S11: eq. 28's f_pre ~ |dF|^-0.9 makes dT depend on dF only through sgn(dF)|dF|^0.1,
                 * so a dF that is pure rounding noise (deep isothermal layers: F_up == F_dn == pi B)
                 * would still kick the layer by O(1 K) with a random sign.  A layer that already meets
                 * eq. 29 locally, |dF_i| < flux_floor * sigma T_i^4, is in equilibrium: dF_i := 0. */
                if (fabs(dF) < p->flux_floor * (sigma * Tc[i] * Tc[i] * Tc[i] * Tc[i])) dF = 0.0;
                dT[i] = orc_re_delta_T(dF, a[i], p_layer[i], p_interface[i] - p_interface[i + 1],
                                       Tc[i], p->dT_frac_max);
                if (fabs(dT[i]) > max_dT) max_dT = fabs(dT[i]);
                const double rel = fabs(dF) / (sigma * Tc[i] * Tc[i] * Tc[i] * Tc[i]);  /* eq. 29 */
                if (rel > max_rel) max_rel = rel;
            }
            if (dT_last) memcpy(dT_last + (size_t)c * n, dT, sizeof(double) * n);
            if ((tol_dT > 0.0 && max_dT < tol_dT) || (tol_flux > 0.0 && max_rel < tol_flux)) {
                conv = 1;
                break;
            }
            for (int i = 0; i < n; ++i) {
                double t = Tc[i] + dT[i];
                if (t < p->T_floor) t = p->T_floor;
                Tc[i] = t;
                h[i] = orc_hist_push(h[i], dT[i]);
                a[i] *= orc_hist_factor(h[i]);
            }
        }
        iters[c] += it;
        converged[c] = conv;
        free(Fu); free(Fd); free(dT);
    }
}

/* ------------------------------------------------------------------------- */
/* Helpers used only by the pins                                             */
/* ------------------------------------------------------------------------- */

/* Exact pure-absorption transmissivity, eq. 6, by direct midpoint-free
 * Gauss-free brute force: composite Simpson on mu in [0,1] with nint panels. */
double orc_exact_transmissivity_quadrature(double dtau, int nint)
{
    /* integrand 2 mu exp(-dtau/mu); -> 0 at mu = 0 */
    double s = 0.0;
    const double hstep = 1.0 / (double)nint;
    for (int i = 0; i <= nint; ++i) {
        const double mu = hstep * (double)i;
        const double f = (mu > 0.0) ? 2.0 * mu * exp(-dtau / mu) : 0.0;
        const double wgt = (i == 0 || i == nint) ? 1.0 : ((i & 1) ? 4.0 : 2.0);
        s += wgt * f;
    }
    return s * hstep / 3.0;
}

/* Exact non-isothermal pure-absorption layer, eq. 4 with the transmissivity
 * `trans` of eq. 6 supplied by the caller; B_src/B_dst labelling as in eq. 4 (source-side B). */
void orc_exact_layer_eq4(double dtau, double trans, double B_lo, double B_up,
                         double F_up_lo, double F_dn_up, double *F_up_up, double *F_dn_lo)
{
    /* eq. 4 is written with B_1 at the lower interface for the upward flux and B_2 at the upper
     * interface for the downward flux, B' = (B_2-B_1)/(tau_2-tau_1) with tau_2 - tau_1 = -dtau
     * (tau decreases upward), i.e. B' = (B_lo - B_up)/dtau as everywhere else in this file. */
    const double Bp = (B_lo - B_up) / dtau;
    const double br = (2.0 / 3.0) * (1.0 - exp(-dtau)) - dtau * (1.0 - trans / 3.0);
    *F_up_up = trans * F_up_lo + ORC_PI * B_lo * (1.0 - trans) + ORC_PI * Bp * br;
    *F_dn_lo = trans * F_dn_up + ORC_PI * B_up * (1.0 - trans) - ORC_PI * Bp * br;
}
