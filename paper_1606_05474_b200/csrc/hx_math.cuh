// hx_math.cuh -- device math of the HELIOS hot path: exponential of a non-positive argument and
// the incomplete Planck integrals.  Product code (CUDA path); shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace hx {

// (hi, lo) += x with the rounding error of hi + x collected in lo (Neumaier / TwoSum, branch-free)
__device__ __forceinline__ void dd_add(double& hi, double& lo, double x)
{
    const double s = hi + x;
    const double bp = s - hi;
    lo += (hi - (s - bp)) + (x - bp);
    hi = s;
}

// Taylor coefficients 1/k!, k = 13..0, in constant memory so that they enter DFMA as constant-bank
// operands instead of being rematerialised into registers at every use.
__constant__ double c_exp_taylor[14] = {
    1.0 / 6227020800.0, 1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0,
    1.0 / 40320.0, 1.0 / 5040.0, 1.0 / 720.0, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0, 0.5, 1.0, 1.0};

// exp(t) for |t| <= 0.35 by its degree-13 Taylor polynomial (truncation 4e-18).
__device__ __forceinline__ double exp_poly13(double t)
{
    double p = c_exp_taylor[0];
#pragma unroll
    for (int k = 1; k < 14; ++k) p = fma(p, t, c_exp_taylor[k]);
    return p;
}

// p * 2^n for p in [0.70, 1.42], n <= 0, through the exponent field (valid for n >= -1021).
__device__ __forceinline__ double scale_pow2(double p, int n)
{
    const int hi = __double2hiint(p) + (n << 20);
    return __hiloint2double(hi, __double2loint(p));
}

// 2^y for y <= 0 (fp64).  y = n + f, n = rint(y), |f| <= 1/2; 2^f = exp(f ln2).  The relative
// error is that of y itself (|y| * 2^-53) plus ~1 ulp.  Results below 2^-1021 are flushed to zero
// (they multiply fluxes of at most ~1e12, so nothing representable is lost); for such y the
// intermediate values are meaningless and discarded by the final select.
__device__ __forceinline__ double exp2_nonpos(double y)
{
    const double kMagic = 6755399441055744.0;   // 1.5 * 2^52
    const double tn = y + kMagic;
    const int n = __double2loint(tn);
    const double f = y - (tn - kMagic);
    const double r = scale_pow2(exp_poly13(f * 0.693147180559945309417232121458), n);
    return (y < -1021.0) ? 0.0 : r;
}

// 2^(y/256) for y <= 0 with a 256-entry table tab[j] = 2^(j/256) (shared memory): y = k + r,
// k = rint(y), |r| <= 1/2; 2^(y/256) = 2^(k>>8) * tab[k&255] * exp(r ln2/256), the last factor by its
// degree-4 Taylor polynomial in r with the powers of ln2/256 folded into the coefficients
// (|r ln2/256| <= 0.00136: truncation 4e-17).  8 DP instructions instead of 18 for the plain version.
// Results below 2^-1021 are flushed to zero.
constexpr int kExpTab = 256;
constexpr double kExpL = 0.693147180559945309417232121458 / kExpTab;
__constant__ double c_exp_tab_poly[4] = {kExpL * kExpL * kExpL * kExpL / 24.0, kExpL * kExpL * kExpL / 6.0,
                                         kExpL * kExpL / 2.0, kExpL};
__device__ __forceinline__ double exp2_nonpos_tab(double y, const double* __restrict__ tab)
{
    const double kMagic = 6755399441055744.0;   // 1.5 * 2^52
    const double tn = y + kMagic;
    const int k = __double2loint(tn);
    const double r = y - (tn - kMagic);
    double p = fma(c_exp_tab_poly[0], r, c_exp_tab_poly[1]);
    p = fma(p, r, c_exp_tab_poly[2]);
    p = fma(p, r, c_exp_tab_poly[3]);
    p = fma(p, r, 1.0);
    const double v = scale_pow2(p * tab[k & (kExpTab - 1)], k >> 8);
    return (y < -1021.0 * kExpTab) ? 0.0 : v;
}

// 1/x for normal, finite x away from the over/underflow range (|x| in [1e-290, 1e290]):
// MUFU.RCP64H seed (2^-23 relative) + two Newton steps; ~1 ulp, no slow-path branch.
__device__ __forceinline__ double rcp_fast(double x)
{
    double r;
#if defined(__CUDA_ARCH__)
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
#else
    r = 1.0 / x;
#endif
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    return r;
}

// e^x for x <= 0 (fp64, ~1 ulp): Cody-Waite reduction x = n ln2 + t with a two-part ln2.
__device__ __forceinline__ double exp_nonpos(double x)
{
    const double kMagic = 6755399441055744.0;
    const double tn = fma(x, 1.44269504088896340735992468100, kMagic);
    const int n = __double2loint(tn);
    const double fn = tn - kMagic;
    double t = fma(fn, -6.93147180369123816490e-01, x);    // ln2 high part (32 trailing zero bits)
    t = fma(fn, -1.90821492927058770002e-10, t);           // ln2 low part
    const double r = scale_pow2(exp_poly13(t), n);
    return (x < -708.0) ? 0.0 : r;
}

// 1/m, m = 0..47 (index 0 unused)
__constant__ double c_inv_m[48] = {
    0.0, 1.0, 1.0 / 2, 1.0 / 3, 1.0 / 4, 1.0 / 5, 1.0 / 6, 1.0 / 7, 1.0 / 8, 1.0 / 9, 1.0 / 10,
    1.0 / 11, 1.0 / 12, 1.0 / 13, 1.0 / 14, 1.0 / 15, 1.0 / 16, 1.0 / 17, 1.0 / 18, 1.0 / 19,
    1.0 / 20, 1.0 / 21, 1.0 / 22, 1.0 / 23, 1.0 / 24, 1.0 / 25, 1.0 / 26, 1.0 / 27, 1.0 / 28,
    1.0 / 29, 1.0 / 30, 1.0 / 31, 1.0 / 32, 1.0 / 33, 1.0 / 34, 1.0 / 35, 1.0 / 36, 1.0 / 37,
    1.0 / 38, 1.0 / 39, 1.0 / 40, 1.0 / 41, 1.0 / 42, 1.0 / 43, 1.0 / 44, 1.0 / 45, 1.0 / 46,
    1.0 / 47};

// Number of terms of the upper series needed at x >= 1 for a relative truncation below 1e-17 (used at
// x >= kPlanckSwitch = 2: at most 21):
// term_m/term_1 ~ e^{-(m-1)x}/m.
__device__ __forceinline__ int planck_upper_terms(double x)
{
    const int m = 2 + (int)(39.2 / x);
    return m > 42 ? 42 : m;
}

// The incomplete Planck integral is taken from the lower (Bernoulli) series below x = kPlanckSwitch and from the upper
// (exponential) series above it.  The upper series needs 2 + 39.2/x terms of ~7 DP instructions each, and a warp
// runs the largest count among its lanes: with the switch at 2 instead of 1 that is at most 21 terms instead of 41,
// for six more (cheap) terms of the lower series.
constexpr double kPlanckSwitch = 2.0;

// Lower incomplete Planck integral H(x) = int_0^x t^3/(e^t-1) dt, 0 <= x < 2:
// t/(e^t-1) = sum_k B_k t^k/k!  =>  H = x^3 [1/3 - x/8 + x^2 sum_j c_j x^(2j)],
// c_j = B_(2j+2)/((2j+2)! (2j+5)), j = 0..15 (B_2 .. B_32; computed in exact rational arithmetic and rounded once).
// Sixteen terms leave 4e-18 relative at x = 2 (the terms fall like (x/2pi)^2 = 0.1), 1e-33 at x = 1.
// Literal coefficients (the compiler keeps them in its constant bank): a __constant__ array here cost the fp64 ray
// kernel 3 % (register allocation at 255 registers), measured.
__device__ __forceinline__ double planck_lower(double x)
{
    const double x2 = x * x;
    double s = -1.641368762534915e-27;
    s = fma(s, x2, 6.87258318890207e-26);
    s = fma(s, x2, -2.888231428076628e-24);
    s = fma(s, x2, 1.2188644964239542e-22);
    s = fma(s, x2, -5.1683202540046385e-21);
    s = fma(s, x2, 2.203601131344092e-19);
    s = fma(s, x2, -9.455950863295921e-18);
    s = fma(s, x2, 4.088600979179926e-16);
    s = fma(s, x2, -1.784042261222412e-14);
    s = fma(s, x2, 7.872080312167458e-13);
    s = fma(s, x2, -3.522793425791662e-11);
    s = fma(s, x2, 1.6059043836821615e-09);
    s = fma(s, x2, -7.515632515632516e-08);
    s = fma(s, x2, 3.6743092298647855e-06);
    s = fma(s, x2, -0.0001984126984126984);
    s = fma(s, x2, 0.016666666666666666);
    s = fma(s, x2, -0.125 * x + 1.0 / 3.0);
    return s * x2 * x;
}

// One term of the upper series  G(x) = int_x^inf t^3/(e^t-1) dt
//   = sum_{m>=1} e^{-m x} (x^3/m + 3x^2/m^2 + 6x/m^3 + 6/m^4);  em = e^{-m x}, rm = 1/m.
__device__ __forceinline__ double planck_upper_term(double x, double x2, double x3, double em,
                                                    double rm)
{
    double q = fma(6.0, rm, 6.0 * x);     // 6x + 6/m
    q = fma(q, rm, 3.0 * x2);
    q = fma(q, rm, x3);
    return em * rm * q;
}

// G(x), x >= 1, with a caller-chosen term count (scalar use: setup-time kernels).
__device__ inline double planck_upper(double x)
{
    const double e1 = exp_nonpos(-x);
    const double x2 = x * x, x3 = x2 * x;
    const int M = planck_upper_terms(x);
    double em = 1.0, s = 0.0;
    for (int m = 1; m <= M; ++m) {
        em *= e1;
        s += planck_upper_term(x, x2, x3, em, c_inv_m[m]);
    }
    return s;
}

// H(2) and G(2) = pi^4/15 - H(2), used when a bin straddles the switch: H(2) from the series above in exact rational
// arithmetic with 22 terms (60-digit evaluation), rounded once.
constexpr double kPlanckH1 = 1.1763425966069978;      // H(kPlanckSwitch)
constexpr double kPlanckG1 = 5.3175968056598313;      // G(kPlanckSwitch)
static_assert(kPlanckSwitch == 2.0, "kPlanckH1 / kPlanckG1 are the values at x = 2");

// Edge value: x < kPlanckSwitch -> -H(x) (sign bit marks the lower branch), x >= kPlanckSwitch -> G(x).
// Bin integral int_{x_lo}^{x_hi} from two edge values (x_lo <= x_hi):
__device__ __forceinline__ double planck_bin_integral(double e_lo, double e_hi)
{
    const bool lo_low = __double2hiint(e_lo) < 0, hi_low = __double2hiint(e_hi) < 0;
    // both lower: H(hi) - H(lo) = e_lo - e_hi (values are negated); both upper: G(lo) - G(hi)
    double r = e_lo - e_hi;
    if (lo_low && !hi_low) r = (kPlanckH1 + e_lo) + (kPlanckG1 - e_hi);
    return r;
}

// Exponential integral E_1(x), x > 0.  x <= 2: -gamma - ln x - sum_k (-x)^k/(k k!), 30 terms
// (2^30/(30 30!) < 2e-25; the alternating terms reach x^2/4 = 1, so the absolute error is ~3e-16);
// x > 2: continued fraction e^-x / (x + 1 - 1/(x + 3 - 4/(x + 5 - 9/(x + 7 - ...)))) evaluated from the
// tail, depth 6 + 110/x (checked against 60-digit arithmetic: relative truncation < 2e-17 for x >= 2).
// Used by the exact pure-absorption mode only (one evaluation per sublayer; not a hot path).
__device__ __forceinline__ double expint_e1(double x)
{
    if (x <= 2.0) {
        double sum = 0.0, term = 1.0;
        for (int k = 1; k <= 30; ++k) {           // 1/k from the constant table: no divisions
            term *= -x * c_inv_m[k];
            sum = fma(-term, c_inv_m[k], sum);
        }
        return -0.57721566490153286060651209008240243 - log(x) + sum;
    }
    const int depth = 6 + (int)(110.0 * rcp_fast(x));
    double f = x + (double)(2 * depth + 1);
    for (int i = depth; i >= 1; --i) f = fma(-(double)(i * i), rcp_fast(f), x + (double)(2 * i - 1));
    return exp_nonpos(-x) * rcp_fast(f);
}

// Transmissivity of eq. 6 and e^-dtau; T(0) = 1.  Not inlined: the callers unroll over the
// lane's sublayers (register arrays), and this mode is not a hot path.
static __device__ __noinline__ double exact_transmissivity(double dtau, double& emd)
{
    emd = exp(-dtau);
    if (!(dtau > 0.0)) return 1.0;
    return fma(1.0 - dtau, emd, dtau * dtau * expint_e1(dtau));
}

}  // namespace hx
