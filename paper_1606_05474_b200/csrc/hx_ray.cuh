// hx_ray.cuh -- one ray (column, bin, g) of the two-stream solve held in the registers of LPR lanes of a warp.
// Product code (CUDA path); shares nothing with oracle/.
//
// Layout.  A warp holds RPW = 32 / LPR rays side by side (LPR = 8, 16 or 32 lanes per ray; the rays of a warp are
// Gauss points of one bin).  The padded column has LPR*S sublayers; sub-lane sl = lane % LPR owns sublayers
// sl*S .. sl*S+S-1 ("local" j = 0..S-1) and the levels sl*S .. sl*S+S-1; level sl*S+S is the next lane's local
// level 0.  Padded sublayers have dtau = 0, for which the coefficients below reduce to the identity map,
// so the TOA boundary value simply travels through them.
//
// Per sublayer (eq. 8, 11-15 with readings G1, G2, G5, S2 of DESIGN.md):
//   F_dn[s]   = a F_dn[s+1] - b F_up[s]   + sd        a = xi/alpha, b = beta/alpha,
//   F_up[s+1] = a F_up[s]   - b F_dn[s+1] + su        sd = S_dn/alpha, su = S_up/alpha
// With the other direction's fluxes frozen, one sweep is an affine recurrence along the column.
// Each lane runs it over its S sublayers from a zero input (which yields the lane's affine map
// (A, C)), the LPR maps of a ray are combined by an exclusive Kogge-Stone scan with warp shuffles of width LPR
// (log2(LPR) dependent shuffle rounds: the first round combines the two nearest neighbours at once), and the
// lane then runs the recurrence once more from its true input.  The products of A the scan needs do not
// depend on the sweep and are formed once per ray.
//
// Why LPR < 32 when the column allows it (100 layers: LPR = 16, S = 13): the scan's shuffle -> DFMA rounds are a
// dependent chain that one warp cannot hide; with two rays per warp every shuffle serves both, there is one
// round fewer, and 200 sublayers fill 208 slots instead of 224.
#pragma once
#include "helios_internal.h"
#include "hx_math.cuh"

namespace hx {

constexpr unsigned kFull = 0xffffffffu;

template <int LPR> struct SegOf {
    static_assert(LPR == 8 || LPR == 16 || LPR == 32, "lanes per ray");
    static constexpr int ROUNDS = LPR == 32 ? 5 : LPR == 16 ? 4 : 3;   // log2(LPR)
    static constexpr int RPW = 32 / LPR;                                 // rays per warp
};

template <int S, int LPR, bool ISO>
struct RayShape {
    static constexpr int NSUB_PAD = LPR * S;
    static constexpr int NN = NSUB_PAD + 1;                 // node slots (levels) incl. the top one
    static constexpr int UP = ISO ? 0 : 1;                  // node offset of a sublayer's upper end
    static constexpr int NACC = ISO ? S : (S + 1) / 2;      // interface accumulators per lane
};

// Accumulators a warp carries over all its (bin, g) rays live in shared memory, one private column
// per lane ([row][lane], conflict-free), so that they do not occupy registers during the sweeps:
//   rows 0..NACC-1        sum w dnu F_up at the lane's interface levels (up-sweep ownership)
//   rows NACC..2NACC-1    sum w dnu F_dn at the lane's interface levels (down-sweep ownership)
//   row 2NACC             F_up at level 0 (BOA); sub-lane 0's is used
//   row 2NACC+1           F_dn at level LPR*S (the boundary value itself); sub-lane LPR-1's is used
//   rows 2NACC+2, +3      per-bin spectra sum_g w_g F_up(TOA) / F_dn(BOA)
// These rows hold the sums over the rays of ONE bin.  COMP (fp64 ray arithmetic): at the end of every bin the
// NF = 2 NACC + 2 flux rows are added to a running double-double sum (rows HI, LO; Neumaier's compensated
// addition) -- the same association as a per-bin sum over g followed by a compensated sum over the bins --
// so that the bolometric sums carry ~1e-17 instead of ~1e-15 relative rounding (the RE
// step turns flux noise into temperature noise).  Without COMP (fp32 ray arithmetic) the flux rows simply
// run on over the bins.
template <int NACC, bool COMP>
struct AccRows {
    static constexpr int UP = 0, DN = NACC, UP0 = 2 * NACC, DNT = 2 * NACC + 1, NF = 2 * NACC + 2,
                         SPU = NF, SPD = NF + 1, HI = NF + 2, LO = HI + NF, ROWS = COMP ? LO + NF : NF + 2;
};

template <int W> __device__ __forceinline__ double shfl_down_w(double v, int d)
{
    const int lo = __shfl_down_sync(kFull, __double2loint(v), d, W);
    const int hi = __shfl_down_sync(kFull, __double2hiint(v), d, W);
    return __hiloint2double(hi, lo);
}
template <int W> __device__ __forceinline__ double shfl_up_w(double v, int d)
{
    const int lo = __shfl_up_sync(kFull, __double2loint(v), d, W);
    const int hi = __shfl_up_sync(kFull, __double2hiint(v), d, W);
    return __hiloint2double(hi, lo);
}
template <int W> __device__ __forceinline__ double shfl_idx_w(double v, int l) { return __shfl_sync(kFull, v, l, W); }
template <int W> __device__ __forceinline__ float shfl_down_w(float v, int d) { return __shfl_down_sync(kFull, v, d, W); }
template <int W> __device__ __forceinline__ float shfl_up_w(float v, int d) { return __shfl_up_sync(kFull, v, d, W); }
template <int W> __device__ __forceinline__ float shfl_idx_w(float v, int l) { return __shfl_sync(kFull, v, l, W); }

// Sublayer coefficients for the lane's S sublayers.  kap points at the lane's first node; Bm / Bh at
// the lane's first sublayer.  PS = the bin is a pure-scattering one (eq. 14); decided once per bin,
// not per sublayer.
// Bm = (2 pi / D) x the mean of the bin-mean Planck function at the sublayer's two ends, Bh = (2 pi / D)
// x half the difference (lower end - upper end); both are staged once per bin (they do not depend on the
// Gauss point).  With w1 = alpha + beta - xi, w2 = alpha + beta + xi, w3 = alpha - xi - beta = 2 alpha - w2,
// eq. 15 (readings G1, G2) with B_lo = Bm + Bh, B_up = Bm - Bh reads
//   S_up = Bm w1 - Bh [w2 - (2 kp / dtau) w3],   S_dn = Bm w1 + Bh [w2 - (2 kp / dtau) w3],
// and eq. 11 (dtau < dtau_iso, reading S2: B = mean of the ends) is the same with Bh = 0.
// WABS: b[j] receives the sublayer's absorptance w = 1 - rho - a = (alpha + beta - xi)/alpha (rho = -beta/alpha
// its reflectance, a its transmittance) instead of beta/alpha: the direct solve works with (a, w), which stay
// accurate when rho -> 1 (near-conservative scattering); w = 0 exactly for eq. 14.
template <int S, bool ISO, bool PS, bool WABS = false>
__device__ __forceinline__ void ray_coefficients(const BinConst& bc, const double* __restrict__ exp_tab,
                                                 double dtau_iso,
                                                 const double* __restrict__ kap,
                                                 const double* __restrict__ hP,
                                                 const double* __restrict__ Bm,
                                                 const double* __restrict__ Bh,
                                                 double (&a)[S], double (&b)[S], double (&su)[S],
                                                 double (&sd)[S])
{
    double k_lo = kap[0];
    const double kp2 = 2.0 * bc.kp;
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const double k_up = ISO ? k_lo : kap[j + 1];
        const double dtau = hP[j] * (k_lo + k_up);                   // eq. 19, kappa = mean of the ends
        if (!PS) {
            const double tr = exp2_nonpos_tab(bc.nlam_tab * dtau, exp_tab);   // eq. 8
            const double om = fma(-tr, tr, 1.0);                    // 1 - T^2
            const double alpha = fma(-bc.zm2, om, -bc.r);           // eq. 12: zm^2 T^2 - zp^2 = (zm^2 - zp^2) - zm^2 (1 - T^2)
            const double beta = bc.zpzm * om;
            const double xi = -bc.r * tr;                           // (zm^2 - zp^2) T = -r T
            const bool thin = !(dtau >= dtau_iso);                  // PAPER.md:232 (dtau_iso > 0)
            const double dsafe = thin ? 1.0 : dtau;
            const double inv = rcp_fast(alpha * dsafe);             // one reciprocal for 1/alpha, 1/dtau
            const double ia = dsafe * inv;
            // the small combinations are formed from alpha, beta, xi themselves (as the oracle's plain forms
            // do) and divided by alpha afterwards: 1 + b - a would carry the rounding of 1/alpha in full
            const double apb = alpha + beta;
            const double w1 = apb - xi, w2 = apb + xi;              // alpha + beta -/+ xi
            const double w3 = fma(2.0, alpha, -w2);                 // alpha - xi - beta
            const double kpi = kp2 * (alpha * inv);                 // 2 eps / ((1 - w0 g0) dtau)   (G2)
            const double G = fma(-kpi, w3, w2) * ia;
            const double E = (thin ? 0.0 : Bh[j]) * G;
            const double wn = w1 * ia;
            const double m = Bm[j] * wn;
            a[j] = xi * ia;
            b[j] = WABS ? wn : beta * ia;
            su[j] = m - E;
            sd[j] = m + E;
        } else {                                                    // eq. 14
            const double x = bc.xfac * dtau;
            const double inv = rcp_fast(2.0 + x);
            a[j] = 2.0 * inv;
            b[j] = WABS ? 0.0 : -x * inv;
            su[j] = 0.0;
            sd[j] = 0.0;
        }
        if (!ISO) k_lo = k_up;
        else if (j + 1 < S) k_lo = kap[j + 1];
    }
}

// Exact pure-absorption limit (params.exact_absorption, S13): no coupling
// (b = 0), a = T of eq. 6, sources of eq. 4 -- pi B_src (1 - T) +/- pi B' {2/3 (1 - e^-dtau) - dtau (1 - T/3)}
// with B' = (B_lo - B_up)/dtau, B_src = B_lo for the upward and B_up for the downward flux -- or of eq. 3
// with B = mean of the ends below dtau_iso (S2).  Bm / Bh hold pi x (mean, half difference) here.
// Evaluated in fp64 whatever the ray arithmetic (E_1, 1 - T), then rounded to T.
template <typename T, int S, bool ISO>
__device__ __forceinline__ void ray_coefficients_exact(double dtau_iso, const T* __restrict__ kap,
                                                       const T* __restrict__ hP, const T* __restrict__ Bm,
                                                       const T* __restrict__ Bh, T (&a)[S], T (&b)[S],
                                                       T (&su)[S], T (&sd)[S])
{
    double k_lo = (double)kap[0];
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const double k_up = ISO ? k_lo : (double)kap[j + 1];
        const double dtau = (double)hP[j] * (k_lo + k_up);           // eq. 19
        double emd;
        const double tr = exact_transmissivity(dtau, emd);           // eq. 6
        const double omt = 1.0 - tr;
        const bool thin = !(dtau >= dtau_iso);
        const double bm = (double)Bm[j], bh = thin ? 0.0 : (double)Bh[j];
        const double br = (2.0 / 3.0) * (1.0 - emd) - dtau * (1.0 - tr * (1.0 / 3.0));
        const double g = thin ? 0.0 : (bh + bh) / dtau * br;         // pi B' {...}
        a[j] = (T)tr;
        b[j] = T(0);
        su[j] = (T)((bm + bh) * omt + g);                            // eq. 4, upward: B_lo
        sd[j] = (T)((bm - bh) * omt - g);                            // eq. 4, downward: B_up
        if (!ISO) k_lo = k_up;
        else if (j + 1 < S) k_lo = (double)kap[j + 1];
    }
}

// Single-scattering albedo per sublayer (helios_set_scattering, S14): a scattering
// opacity ksc of the bin is added to the table opacity at every node and w0 = ksc / (mean total opacity of the
// sublayer), so lambda, zeta_+-, r and eps/(1 - w0 g0) of eq. 8, 12-13, 15 -- per-bin constants otherwise --
// are formed per sublayer here, as is the switch to eq. 14 "in this layer and waveband".  Always in fp64, rounded
// to T at the end.  Same devices as ray_coefficients: the table exp2, branch-free reciprocals (three per sublayer:
// 1/(k_lo + k_up), 1/(1 - w0 g0) and the shared 1/(alpha dtau)), one square root (lambda' = sqrt((1 - w0)(1 - w0 g0));
// r = sqrt((1 - w0)/(1 - w0 g0)) = lambda'/(1 - w0 g0)), alpha = -(r + zeta_-^2 (1 - T^2)) since
// zeta_-^2 - zeta_+^2 = -r.  Bm / Bh as for ray_coefficients.
template <typename T, int S, bool ISO, bool WABS>
__device__ __forceinline__ void ray_coefficients_w0s(double D, double g0, double ksc, double dtau_iso,
                                                     double omw_min, const double* __restrict__ exp_tab,
                                                     const T* __restrict__ kap,
                                                     const T* __restrict__ hP, const T* __restrict__ Bm,
                                                     const T* __restrict__ Bh, T (&a)[S], T (&b)[S],
                                                     T (&su)[S], T (&sd)[S])
{
    const double nDl = -D * (1.44269504088896340735992468100 * kExpTab);   // tr = 2^(nDl lambda' dtau / 256)
    const double two_eps = 2.0 / D, xfac = D * (1.0 - g0), ksc2 = ksc + ksc;
    double k_lo = (double)kap[0] + ksc;
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const double k_up = ISO ? k_lo : (double)kap[j + 1] + ksc;
        const double ksum = k_lo + k_up;
        const double dtau = (double)hP[j] * ksum;                    // eq. 19 with the total opacity
        const bool has = ksum > 0.0;
        const double w0 = has ? ksc2 * rcp_fast(has ? ksum : 1.0) : 0.0;             // ksc / (mean opacity)
        const double u = 1.0 - w0;
        double aj, bj, suj = 0.0, sdj = 0.0;
        if (u < omw_min) {                                           // eq. 14
            const double x = xfac * dtau;
            const double inv = rcp_fast(2.0 + x);
            aj = 2.0 * inv;
            bj = WABS ? 0.0 : -x * inv;
        } else {
            const double q = fma(-w0, g0, 1.0);                      // 1 - w0 g0
            const double iq = rcp_fast(q);
            const double lam = sqrt(q * u);                          // lambda / D
            const double r = lam * iq;                               // sqrt((1 - w0)/(1 - w0 g0))
            const double zp = 0.5 * (1.0 + r), zm = 0.5 * (1.0 - r);                 // eq. 13
            const double tr = exp2_nonpos_tab(nDl * lam * dtau, exp_tab);            // eq. 8
            const double om = fma(-tr, tr, 1.0);
            const double alpha = fma(-(zm * zm), om, -r);            // eq. 12
            const double beta = zp * zm * om;
            const double xi = -r * tr;
            const bool thin = !(dtau >= dtau_iso);
            const double dsafe = thin ? 1.0 : dtau;
            const double inv = rcp_fast(alpha * dsafe);              // one reciprocal for 1/alpha, 1/dtau
            const double ia = dsafe * inv;
            const double apb = alpha + beta;
            const double w1 = apb - xi, w2 = apb + xi, w3 = fma(2.0, alpha, -w2);
            const double kpi = two_eps * iq * (alpha * inv);         // 2 eps / ((1 - w0 g0) dtau)  (G2)
            const double G = fma(-kpi, w3, w2) * ia;
            const double E = (thin ? 0.0 : (double)Bh[j]) * G;
            const double wn = w1 * ia;
            const double m = (double)Bm[j] * wn;
            aj = xi * ia;
            bj = WABS ? wn : beta * ia;
            suj = m - E;
            sdj = m + E;
        }
        a[j] = (T)aj;
        b[j] = (T)bj;
        su[j] = (T)suj;
        sd[j] = (T)sdj;
        if (!ISO) k_lo = k_up;
        else if (j + 1 < S) k_lo = (double)kap[j + 1] + ksc;
    }
}

// Tabulated transmission function (params.trans_table_dlog10k, S16): for one bin and one
// sublayer eq. 8 is a function of the opacity alone, T(kappa) = exp(-c kappa), c = lambda dtau / kappa; the table's
// nodes are kappa_k = 10^(k dlog) and the value is linear in log10 kappa between two nodes.  The two node values are
// evaluated on the fly (what a stored table would hold: on B200 the exact exp2 of ray_coefficients costs 8 DP
// instructions, less than the table look-up's log10, so this mode is an approximation kept for parity with the
// paper's option, not a fast path).  Everything else as in ray_coefficients, plain forms in fp64, rounded to T.
template <typename T, int S, bool ISO, bool PS, bool WABS>
__device__ __forceinline__ void ray_coefficients_tt(const BinConst& bc, double dlog, double dtau_iso,
                                                    const T* __restrict__ kap, const T* __restrict__ hP,
                                                    const T* __restrict__ Bm, const T* __restrict__ Bh,
                                                    T (&a)[S], T (&b)[S], T (&su)[S], T (&sd)[S])
{
    double k_lo = (double)kap[0];
    const double inv_dlog = 1.0 / dlog;
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const double k_up = ISO ? k_lo : (double)kap[j + 1];
        const double ksum = k_lo + k_up;
        const double dtau = (double)hP[j] * ksum;                    // eq. 19
        double aj, bj, suj = 0.0, sdj = 0.0;
        if (PS) {                                                    // eq. 14: no transmission function
            const double x = bc.xfac * dtau;
            const double inv = 1.0 / (2.0 + x);
            aj = 2.0 * inv;
            bj = WABS ? 0.0 : -x * inv;
        } else {
            const double kbar = 0.5 * ksum;
            double tr = 1.0;
            if (kbar > 0.0) {
                const double c = bc.lam * dtau / kbar;
                const double u = log10(kbar) * inv_dlog;
                const double k = floor(u);
                const double t0 = exp(-c * exp10(k * dlog)), t1 = exp(-c * exp10((k + 1.0) * dlog));
                tr = fma(u - k, t1 - t0, t0);
            }
            const double om = fma(-tr, tr, 1.0);
            const double alpha = bc.zm2 * tr * tr - bc.zp2;          // eq. 12
            const double beta = bc.zpzm * om;
            const double xi = -bc.r * tr;
            const double ia = 1.0 / alpha;
            const bool thin = !(dtau >= dtau_iso);
            const double apb = alpha + beta;
            const double w1 = apb - xi, w2 = apb + xi, w3 = fma(2.0, alpha, -w2);
            const double kpi = thin ? 0.0 : 2.0 * bc.kp / dtau;      // 2 eps / ((1 - w0 g0) dtau)  (G2)
            const double G = fma(-kpi, w3, w2) * ia;
            const double E = (thin ? 0.0 : (double)Bh[j]) * G;
            const double wn = w1 * ia;
            const double m = (double)Bm[j] * wn;
            aj = xi * ia;
            bj = WABS ? wn : beta * ia;
            suj = m - E;
            sdj = m + E;
        }
        a[j] = (T)aj;
        b[j] = (T)bj;
        su[j] = (T)suj;
        sd[j] = (T)sdj;
        if (!ISO) k_lo = k_up;
        else if (j + 1 < S) k_lo = (double)kap[j + 1];
    }
}

// fp32 ray arithmetic (HELIOS_PREC_FP32): the same coefficients in cancellation-free form
// (S3), because 1 - T, alpha + beta - xi and alpha - xi - beta lose all digits in fp32 for
// thin sublayers when formed by subtraction:
//   u = 1 - T = -expm1(-x), x = lambda dtau (series below x = 0.25);  d1 = zeta_+ - zeta_- T;
//   d2 = zeta_+ + zeta_- T;  alpha = -d1 d2;  beta = zeta_+ zeta_- u (1 + T);  xi = -r T;
//   alpha + beta - xi = -u r d1;  alpha - xi - beta = -u d2;
//   S_up = -[u r d1 B_dst + (B_src - B_dst)(xi + kp u d2 / dtau)],  S_dn = -[u r d1 B_src - (...)].
// ex2.approx / rcp.approx (MUFU) are accurate to ~2^-22, within the 1e-4 bar of this path.
__device__ __forceinline__ float ex2_approx(float x)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

template <int S, bool ISO, bool PS, bool WABS = false>
__device__ __forceinline__ void ray_coefficients_f32(const BinConstF& bc, float dtau_iso,
                                                     const float* __restrict__ kap,
                                                     const float* __restrict__ hP,
                                                     const float* __restrict__ Bm,
                                                     const float* __restrict__ Bh,
                                                     float (&a)[S], float (&b)[S], float (&su)[S],
                                                     float (&sd)[S])
{
    float k_lo = kap[0];
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const float k_up = ISO ? k_lo : kap[j + 1];
        const float dtau = hP[j] * (k_lo + k_up);                    // eq. 19
        if (!PS) {
            const float x = bc.lam * dtau;
            const float tr = ex2_approx(bc.nlam2 * dtau);            // eq. 8
            float us = fmaf(x, 1.0f / 5040.0f, -1.0f / 720.0f);      // x - x^2/2 + ... + x^7/5040
            us = fmaf(us, x, 1.0f / 120.0f);
            us = fmaf(us, x, -1.0f / 24.0f);
            us = fmaf(us, x, 1.0f / 6.0f);
            us = fmaf(us, x, -0.5f);
            us = fmaf(us, x, 1.0f);
            us *= x;
            const float u = (x < 0.25f) ? us : 1.0f - tr;
            const float zmT = bc.zm * tr;
            // zeta_+ - zeta_- T = (u + r (1 + T)) / 2: no cancellation when r -> 0 (w0 -> 1) and T -> 1
            const float d1 = 0.5f * fmaf(bc.r, 1.0f + tr, u), d2 = bc.zp + zmT;
            const float alpha = -d1 * d2;                            // eq. 12, factorised
            const float beta = bc.zpzm * u * (1.0f + tr);
            const float xi = -bc.r * tr;
            const bool thin = !(dtau >= dtau_iso);
            const float ia = rcp_approx(alpha);
            const float idt = thin ? 0.0f : rcp_approx(dtau);
            const float bh = thin ? 0.0f : Bh[j];                    // eq. 11 (S2) below dtau_iso: B = mean
            const float Bd = Bm[j] - bh, Bs = Bm[j] + bh;            // B at the upper / lower end
            const float e = u * bc.r * d1;                           // -(alpha + beta - xi)
            const float w = fmaf(bc.kp * u * d2, idt, xi);           // xi + kp u d2 / dtau   (G2)
            const float dw = (bh + bh) * w;
            a[j] = (x == 0.0f) ? 1.0f : xi * ia;            // zero thickness (padding): the identity map exactly
            b[j] = WABS ? -e * ia : beta * ia;
            su[j] = -fmaf(e, Bd, dw) * ia;                           // eq. 15 (G1)
            sd[j] = -fmaf(e, Bs, -dw) * ia;
        } else {                                                     // eq. 14
            const float x = bc.xfac * dtau;
            const float inv = rcp_approx(2.0f + x);
            a[j] = 2.0f * inv;
            b[j] = WABS ? 0.0f : -x * inv;
            su[j] = 0.0f;
            sd[j] = 0.0f;
        }
        if (!ISO) k_lo = k_up;
        else if (j + 1 < S) k_lo = kap[j + 1];
    }
}

// Sweep-independent factors of the exclusive scan of one ray, per direction ("after" = the lanes the flux
// comes from: higher sub-lanes for the down sweep, lower ones for the up sweep); A = product of a over a lane:
//   d[0] / u[0]          A of the neighbouring lane (0 if there is no lane after it)
//   d[k] / u[k], k >= 1  product of A over the 2^k lanes after this one (0 if there is nothing beyond them)
//   d[R] / u[R]          product of A over all lanes after this one (1 on the end lane)
// PL, PH: the two half products of the lane's own sublayers.  The zeros remove every select from the scan rounds.
template <typename T, int LPR>
struct ScanF {
    static constexpr int R = SegOf<LPR>::ROUNDS;
    T d[R + 1], u[R + 1];
    T PL, PH;    // prod a[0 .. H-1], prod a[H .. S-1]
};

// The shuffle part of scan_factors: from the lane's two half products.
template <typename T, int LPR>
__device__ __forceinline__ void scan_factors_from(T PL, T PH, bool two_halves, int sl, ScanF<T, LPR>& F);

template <typename T, int S, int LPR>
__device__ __forceinline__ void scan_factors(const T (&a)[S], int sl, ScanF<T, LPR>& F)
{
    constexpr int H = (S + 1) / 2;
    T PL = a[0], PH = a[H < S ? H : 0];
#pragma unroll
    for (int j = 1; j < H; ++j) PL *= a[j];
#pragma unroll
    for (int j = H + 1; j < S; ++j) PH *= a[j];
    scan_factors_from<T, LPR>(PL, PH, H < S, sl, F);
}

template <typename T, int LPR>
__device__ __forceinline__ void scan_factors_from(T PL, T PH, bool two_halves, int sl, ScanF<T, LPR>& F)
{
    constexpr int R = SegOf<LPR>::ROUNDS;
    F.PL = PL;
    F.PH = PH;
    const T AL = two_halves ? PL * PH : PL;
    T gd = shfl_down_w<LPR>(AL, 1), gu = shfl_up_w<LPR>(AL, 1);     // A of the neighbour
    const bool h1d = sl + 1 < LPR, h1u = sl >= 1;
    gd = h1d ? gd : T(1);
    gu = h1u ? gu : T(1);
    F.d[0] = (sl + 2 < LPR) ? gd : T(0);
    F.u[0] = (sl >= 2) ? gu : T(0);
    // pd / pu: product of A over the 2^k lanes after this one (those that exist)
    const T od1 = shfl_down_w<LPR>(gd, 1), ou1 = shfl_up_w<LPR>(gu, 1);
    T pd = gd * (h1d ? od1 : T(1)), pu = gu * (h1u ? ou1 : T(1));
#pragma unroll
    for (int k = 1; k < R; ++k) {
        const int dd = 1 << k;
        F.d[k] = (sl + dd + 1 < LPR) ? pd : T(0);
        F.u[k] = (sl >= dd + 1) ? pu : T(0);
        const T od = shfl_down_w<LPR>(pd, dd), ou = shfl_up_w<LPR>(pu, dd);
        pd *= (sl + dd < LPR) ? od : T(1);
        pu *= (sl >= dd) ? ou : T(1);
    }
    F.d[R] = pd;
    F.u[R] = pu;
}

// Exclusive scan of the lanes' affine maps: `run` = the lane's zero-input result; returns the flux entering this
// lane (F_dn at its local level S for DOWN, F_up at its local level 0 otherwise), given the boundary value that
// enters the end lane (eq. 20 above sub-lane LPR-1, eq. 22 below sub-lane 0).  log2(LPR) dependent shuffle rounds.
template <typename T, int LPR, bool DOWN>
__device__ __forceinline__ T scan_exclusive(T run, const T (&f)[SegOf<LPR>::ROUNDS + 1], T boundary, int sl)
{
    constexpr int R = SegOf<LPR>::ROUNDS;
    const T c1 = DOWN ? shfl_down_w<LPR>(run, 1) : shfl_up_w<LPR>(run, 1);
    const T c2 = DOWN ? shfl_down_w<LPR>(run, 2) : shfl_up_w<LPR>(run, 2);
    T t = fma(f[0], c2, c1);
    t = (sl == (DOWN ? LPR - 1 : 0)) ? T(0) : t;                // nothing after the end lane
#pragma unroll
    for (int k = 1; k < R; ++k) t = fma(f[k], DOWN ? shfl_down_w<LPR>(t, 1 << k) : shfl_up_w<LPR>(t, 1 << k), t);
    return fma(f[R], boundary, t);
}

// The lane's S sublayers are run as two independent chains, [0, H) and [H, S) with H = (S+1)/2: the zero-input
// run combines them with the half product (run = P_first_half_crossed * r_far + r_near), and after the scan the
// near half starts from F at local level H formed directly as P_far * q + r_far instead of waiting for the far
// chain.  Two more FMAs per sweep, but the dependent DFMA chain of a sweep shrinks from 2S to S + 2.
// One (down sweep, BOA condition, up sweep) pass.  On entry Y[j] = F_up at local level j+1 and
// o0 = F_up at local level 0 (the lane below's Y[S-1]; F_up at level 0 on sub-lane 0); on exit the same
// for the new pass.  FIRST: the upward fluxes are all zero ("starting with the coupled dependencies
// as zero").  LAST: add the interface fluxes, weighted by wq, to the lane's accumulator
// column `acc` (stride 32 doubles per row).  The value a scan hands to a lane (the neighbour's
// boundary flux) is also the "other direction" flux the next sweep needs at that level.
template <typename T, int S, int LPR, bool ISO, bool FIRST, bool LAST>
__device__ __forceinline__ void ray_pass(const T (&a)[S], const T (&b)[S],
                                         const T (&su)[S], const T (&sd)[S],
                                         const ScanF<T, LPR>& F,
                                         T (&Y)[S], T& o0, T& fu0, T& fd0,
                                         T F_top, T piB_int, double wq, int sl,
                                         bool base_odd, double* __restrict__ acc)
{
    constexpr int NACC = RayShape<S, LPR, ISO>::NACC;
    using R = AccRows<NACC, false>;
    constexpr int H = (S + 1) / 2;                         // halves [0, H) and [H, S) run as two chains
    constexpr bool SPLIT = S >= 4;
    T oS;                                                  // F_dn at local level S
    // ---- down sweep: Y[j-1] holds F_up at local level j, o0 at local level 0
    {
#pragma unroll
        for (int j = S - 1; j >= 0; --j) {
            const T other = (j > 0) ? Y[j > 0 ? j - 1 : 0] : o0;
            Y[j] = FIRST ? sd[j] : fma(-b[j], other, sd[j]);
        }
        T run, r_hi = T(0);
        if (SPLIT) {
            r_hi = Y[S - 1];
#pragma unroll
            for (int j = S - 2; j >= H; --j) r_hi = fma(a[j], r_hi, Y[j]);
            T r_lo = Y[H - 1];
#pragma unroll
            for (int j = H - 2; j >= 0; --j) r_lo = fma(a[j], r_lo, Y[j]);
            run = fma(F.PL, r_hi, r_lo);
        } else {
            run = Y[S - 1];
#pragma unroll
            for (int j = S - 2; j >= 0; --j) run = fma(a[j], run, Y[j]);
        }
        const T q = scan_exclusive<T, LPR, true>(run, F.d, F_top, sl);   // eq. 20 enters above the top lane
        oS = q;
        if (SPLIT) {
            const T yb = fma(F.PH, q, r_hi);               // F_dn at local level H, without waiting for the upper chain
            Y[S - 1] = fma(a[S - 1], q, Y[S - 1]);
#pragma unroll
            for (int j = S - 2; j >= H; --j) Y[j] = fma(a[j], Y[j + 1], Y[j]);
            Y[H - 1] = fma(a[H - 1], yb, Y[H - 1]);
#pragma unroll
            for (int j = H - 2; j >= 0; --j) Y[j] = fma(a[j], Y[j + 1], Y[j]);
        } else {
            Y[S - 1] = fma(a[S - 1], q, Y[S - 1]);
#pragma unroll
            for (int j = S - 2; j >= 0; --j) Y[j] = fma(a[j], Y[j + 1], Y[j]);
        }
        fd0 = shfl_idx_w<LPR>(Y[0], 0);
        fu0 = fd0 + piB_int;                                    // eq. 22
    }
    if (LAST) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
            T v;
            if (ISO) v = Y[k];
            else {
                const T ve = Y[(2 * k < S) ? 2 * k : 0];
                const T vo = (2 * k + 1 < S) ? Y[(2 * k + 1 < S) ? 2 * k + 1 : 0] : T(0);
                v = base_odd ? vo : ve;
            }
            acc[32 * (R::DN + k)] = fma(wq, (double)v, acc[32 * (R::DN + k)]);
        }
    }
    // ---- up sweep: Y[j+1] holds F_dn at local level j+1, oS at local level S
    {
#pragma unroll
        for (int j = 0; j < S; ++j) {
            const T other = (j + 1 < S) ? Y[(j + 1 < S) ? j + 1 : 0] : oS;
            Y[j] = fma(-b[j], other, su[j]);
        }
        T run, r_lo = T(0);
        if (SPLIT) {
            r_lo = Y[0];
#pragma unroll
            for (int j = 1; j < H; ++j) r_lo = fma(a[j], r_lo, Y[j]);
            T r_hi = Y[H < S ? H : 0];
#pragma unroll
            for (int j = H + 1; j < S; ++j) r_hi = fma(a[j], r_hi, Y[j]);
            run = fma(F.PH, r_lo, r_hi);
        } else {
            run = Y[0];
#pragma unroll
            for (int j = 1; j < S; ++j) run = fma(a[j], run, Y[j]);
        }
        const T q = scan_exclusive<T, LPR, false>(run, F.u, fu0, sl);    // eq. 22 enters below sub-lane 0
        o0 = q;
        if (SPLIT) {
            const T yb = fma(F.PL, q, r_lo);               // F_up at local level H
            Y[0] = fma(a[0], q, Y[0]);
#pragma unroll
            for (int j = 1; j < H; ++j) Y[j] = fma(a[j], Y[j - 1], Y[j]);
            Y[H < S ? H : 0] = fma(a[H < S ? H : 0], yb, Y[H < S ? H : 0]);
#pragma unroll
            for (int j = H + 1; j < S; ++j) Y[j] = fma(a[j], Y[j - 1], Y[j]);
        } else {
            Y[0] = fma(a[0], q, Y[0]);
#pragma unroll
            for (int j = 1; j < S; ++j) Y[j] = fma(a[j], Y[j - 1], Y[j]);
        }
    }
    if (LAST) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
            T v;
            if (ISO) v = Y[k];
            else {
                // level base + j + 1 even: j = 2k+1 for an even base, j = 2k for an odd base
                const T ve = (2 * k + 1 < S) ? Y[(2 * k + 1 < S) ? 2 * k + 1 : 0] : T(0);
                const T vo = Y[(2 * k < S) ? 2 * k : 0];
                v = base_odd ? vo : ve;
            }
            acc[32 * (R::UP + k)] = fma(wq, (double)v, acc[32 * (R::UP + k)]);
        }
        acc[32 * R::UP0] = fma(wq, (double)fu0, acc[32 * R::UP0]);
        acc[32 * R::DNT] = fma(wq, (double)F_top, acc[32 * R::DNT]);
    }
}

// ---------------------------------------------------------------------------------------------
// fp32 rays with packed arithmetic (sm_100: add / mul / fma.rn.f32x2, SASS FADD2 / FMUL2 / FFMA2 -- one issue slot for
// two operations at the FP32 pipe's flop rate).  The two halves of a lane's sublayers, [0, H) and
// [H, S), go through the same instruction sequence on independent data, so sublayers j and j + H share a register
// pair: X2[j] = (X[j], X[j+H]), j = 0 .. H-1.  For odd S the missing partner (index S) is a zero-thickness sublayer,
// i.e. the identity map (a = 1, b = 0, no source).  Same formulas and the same rounding per component as
// ray_coefficients_f32 / ray_pass<float, ...> (the packed instructions round like the scalar ones).
template <int S>
struct Packed2 {
    static constexpr int H = (S + 1) / 2;
    float2 a[H], b[H], su[H], sd[H];
};
__device__ __forceinline__ float2 f2(float x) { return make_float2(x, x); }
__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }
// element `j` (0 .. S-1) of a packed array
template <int H> __device__ __forceinline__ float p2_get(const float2 (&Y)[H], int j) { return j < H ? Y[j < H ? j : 0].x : Y[j >= H ? j - H : 0].y; }

template <int S, bool ISO, bool WABS>
__device__ __forceinline__ void ray_coefficients_f32_p2(const BinConstF& bc, float dtau_iso,
                                                        const float* __restrict__ kap, const float* __restrict__ hP,
                                                        const float* __restrict__ Bm, const float* __restrict__ Bh,
                                                        Packed2<S>& C)
{
    constexpr int H = (S + 1) / 2;
    const float2 lam = f2(bc.lam), nlam2 = f2(bc.nlam2), zp = f2(bc.zp), zm = f2(bc.zm), zpzm = f2(bc.zpzm), r = f2(bc.r),
                 nr = f2(-bc.r), kp = f2(bc.kp);
#pragma unroll
    for (int j = 0; j < H; ++j) {
        const bool has = j + H < S;                      // compile time after unrolling
        const int jj = has ? j + H : j;
        const float2 k_lo = make_float2(kap[j], kap[jj]);
        const float2 k_up = ISO ? k_lo : make_float2(kap[j + 1], kap[jj + 1]);
        const float2 hp = make_float2(hP[j], has ? hP[jj] : 0.0f);        // the missing partner has zero thickness
        const float2 dtau = __fmul2_rn(hp, __fadd2_rn(k_lo, k_up));       // eq. 19
        const float2 x = __fmul2_rn(lam, dtau);
        const float2 y = __fmul2_rn(nlam2, dtau);
        const float2 tr = make_float2(ex2_approx(y.x), ex2_approx(y.y));  // eq. 8
        float2 us = __ffma2_rn(x, f2(1.0f / 5040.0f), f2(-1.0f / 720.0f));   // x - x^2/2 + ... + x^7/5040
        us = __ffma2_rn(us, x, f2(1.0f / 120.0f));
        us = __ffma2_rn(us, x, f2(-1.0f / 24.0f));
        us = __ffma2_rn(us, x, f2(1.0f / 6.0f));
        us = __ffma2_rn(us, x, f2(-0.5f));
        us = __ffma2_rn(us, x, f2(1.0f));
        us = __fmul2_rn(us, x);
        const float2 omt = __fadd2_rn(f2(1.0f), neg2(tr));
        const float2 u = make_float2(x.x < 0.25f ? us.x : omt.x, x.y < 0.25f ? us.y : omt.y);
        const float2 opt = __fadd2_rn(f2(1.0f), tr);
        const float2 d1 = __fmul2_rn(f2(0.5f), __ffma2_rn(r, opt, u)), d2 = __ffma2_rn(zm, tr, zp);
        const float2 alpha = __fmul2_rn(neg2(d1), d2);                    // eq. 12, factorised
        const float2 beta = __fmul2_rn(__fmul2_rn(zpzm, u), opt);
        const float2 xi = __fmul2_rn(nr, tr);
        const bool thin_x = !(dtau.x >= dtau_iso), thin_y = !(dtau.y >= dtau_iso);
        const float2 ia = make_float2(rcp_approx(alpha.x), rcp_approx(alpha.y));
        const float2 idt = make_float2(thin_x ? 0.0f : rcp_approx(dtau.x), thin_y ? 0.0f : rcp_approx(dtau.y));
        const float2 bh = make_float2(thin_x ? 0.0f : Bh[j], thin_y ? 0.0f : Bh[jj]);   // eq. 11 (S2) below dtau_iso
        const float2 bm = make_float2(Bm[j], Bm[jj]);
        const float2 Bd = __fadd2_rn(bm, neg2(bh)), Bs = __fadd2_rn(bm, bh);
        const float2 e = __fmul2_rn(__fmul2_rn(u, r), d1);               // -(alpha + beta - xi)
        const float2 w = __ffma2_rn(__fmul2_rn(__fmul2_rn(kp, u), d2), idt, xi);   // xi + kp u d2 / dtau   (G2)
        const float2 dw = __fmul2_rn(__fadd2_rn(bh, bh), w);
        const float2 nia = neg2(ia);
        const float2 av = __fmul2_rn(xi, ia);
        C.a[j] = make_float2(x.x == 0.0f ? 1.0f : av.x, x.y == 0.0f ? 1.0f : av.y);   // zero thickness: the identity exactly
        C.b[j] = WABS ? __fmul2_rn(e, nia) : __fmul2_rn(beta, ia);
        C.su[j] = __fmul2_rn(__ffma2_rn(e, Bd, dw), nia);               // eq. 15 (G1)
        C.sd[j] = __fmul2_rn(__ffma2_rn(e, Bs, neg2(dw)), nia);
    }
}

template <int S, int LPR, bool ISO, bool FIRST, bool LAST>
__device__ __forceinline__ void ray_pass_p2(const Packed2<S>& C, const ScanF<float, LPR>& F, float2 (&Y)[(S + 1) / 2],
                                            float& o0, float& fu0, float& fd0, float F_top, float piB_int, double wq,
                                            int sl, bool base_odd, double* __restrict__ acc)
{
    constexpr int NACC = RayShape<S, LPR, ISO>::NACC;
    using R = AccRows<NACC, false>;
    constexpr int H = (S + 1) / 2;
    static_assert(S >= 2, "packed sweeps need two half chains");
    float oS;
    // ---- down sweep: element j-1 holds F_up at local level j, o0 at local level 0
    {
        const float yH = Y[H - 1].x;                            // F_up at local level H, before it is overwritten
#pragma unroll
        for (int j = H - 1; j >= 1; --j) Y[j] = FIRST ? C.sd[j] : __ffma2_rn(neg2(C.b[j]), Y[j - 1], C.sd[j]);
        Y[0] = FIRST ? C.sd[0] : __ffma2_rn(neg2(C.b[0]), make_float2(o0, yH), C.sd[0]);
        float2 r = Y[H - 1];                                    // (r_lo, r_hi): zero-input runs of the two halves
#pragma unroll
        for (int j = H - 2; j >= 0; --j) r = __ffma2_rn(C.a[j], r, Y[j]);
        const float run = fmaf(F.PL, r.y, r.x);
        const float q = scan_exclusive<float, LPR, true>(run, F.d, F_top, sl);   // eq. 20 enters above the top lane
        oS = q;
        const float yb = fmaf(F.PH, q, r.y);                    // F_dn at local level H
        Y[H - 1] = __ffma2_rn(C.a[H - 1], make_float2(yb, q), Y[H - 1]);
#pragma unroll
        for (int j = H - 2; j >= 0; --j) Y[j] = __ffma2_rn(C.a[j], Y[j + 1], Y[j]);
        fd0 = shfl_idx_w<LPR>(Y[0].x, 0);
        fu0 = fd0 + piB_int;                                    // eq. 22
    }
    if (LAST) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
            float v;
            if (ISO) v = p2_get<H>(Y, k);
            else {
                const float ve = p2_get<H>(Y, (2 * k < S) ? 2 * k : 0);
                const float vo = (2 * k + 1 < S) ? p2_get<H>(Y, (2 * k + 1 < S) ? 2 * k + 1 : 0) : 0.0f;
                v = base_odd ? vo : ve;
            }
            acc[32 * (R::DN + k)] = fma(wq, (double)v, acc[32 * (R::DN + k)]);
        }
    }
    // ---- up sweep: element j+1 holds F_dn at local level j+1, oS at local level S
    {
        const float yH = Y[0].y;                                // F_dn at local level H
#pragma unroll
        for (int j = 0; j < H - 1; ++j) Y[j] = __ffma2_rn(neg2(C.b[j]), Y[j + 1], C.su[j]);
        Y[H - 1] = __ffma2_rn(neg2(C.b[H - 1]), make_float2(yH, oS), C.su[H - 1]);
        float2 r = Y[0];
#pragma unroll
        for (int j = 1; j < H; ++j) r = __ffma2_rn(C.a[j], r, Y[j]);
        const float run = fmaf(F.PH, r.x, r.y);
        const float q = scan_exclusive<float, LPR, false>(run, F.u, fu0, sl);    // eq. 22 enters below sub-lane 0
        o0 = q;
        const float yb = fmaf(F.PL, q, r.x);                    // F_up at local level H
        Y[0] = __ffma2_rn(C.a[0], make_float2(q, yb), Y[0]);
#pragma unroll
        for (int j = 1; j < H; ++j) Y[j] = __ffma2_rn(C.a[j], Y[j - 1], Y[j]);
    }
    if (LAST) {
#pragma unroll
        for (int k = 0; k < NACC; ++k) {
            float v;
            if (ISO) v = p2_get<H>(Y, k);
            else {
                const float ve = (2 * k + 1 < S) ? p2_get<H>(Y, (2 * k + 1 < S) ? 2 * k + 1 : 0) : 0.0f;
                const float vo = p2_get<H>(Y, (2 * k < S) ? 2 * k : 0);
                v = base_odd ? vo : ve;
            }
            acc[32 * (R::UP + k)] = fma(wq, (double)v, acc[32 * (R::UP + k)]);
        }
        acc[32 * R::UP0] = fma(wq, (double)fu0, acc[32 * R::UP0]);
        acc[32 * R::DNT] = fma(wq, (double)F_top, acc[32 * R::DNT]);
    }
}

// ray_sweeps for packed fp32 coefficients (cold start only: the warm-start path keeps the scalar form).
template <int S, int LPR, bool ISO>
__device__ __forceinline__ void ray_sweeps_p2(const Packed2<S>& C, float F_top, float piB_int, int n_sweeps,
                                              double wq, double wg, int sl, bool base_odd, int j_top,
                                              bool want_spec, double* __restrict__ acc)
{
    using R = AccRows<RayShape<S, LPR, ISO>::NACC, false>;
    constexpr int H = (S + 1) / 2;
    float2 P = C.a[0];
#pragma unroll
    for (int j = 1; j < H; ++j) P = __fmul2_rn(P, C.a[j]);     // (PL, PH); the identity partner contributes 1
    ScanF<float, LPR> F;
    scan_factors_from<float, LPR>(P.x, P.y, true, sl, F);
    float2 Y[H];
#pragma unroll
    for (int j = 0; j < H; ++j) Y[j] = make_float2(0.0f, 0.0f);
    float fu0 = 0.0f, fd0 = 0.0f, o0 = 0.0f;
    if (n_sweeps == 1) {
        ray_pass_p2<S, LPR, ISO, true, true>(C, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
    } else {
        ray_pass_p2<S, LPR, ISO, true, false>(C, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
        for (int sw = 2; sw < n_sweeps; ++sw)
            ray_pass_p2<S, LPR, ISO, false, false>(C, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
        ray_pass_p2<S, LPR, ISO, false, true>(C, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
    }
    if (want_spec) {
        float ft = 0.0f;
#pragma unroll
        for (int j = 0; j < S; ++j) ft = (j == j_top) ? p2_get<H>(Y, j) : ft;
        acc[32 * R::SPU] = fma(wg, (double)ft, acc[32 * R::SPU]);
        acc[32 * R::SPD] = fma(wg, (double)fd0, acc[32 * R::SPD]);
    }
}

// Runs n_sweeps x (down sweep, BOA condition, up sweep) for one ray and adds the final pass's
// interface fluxes, weighted by wq = w_g * dnu, to the lane's accumulator column.  want_spec: also
// add w_g * F_dn(level 0) and, on the lane that holds it, w_g * F_up(TOA) to the spectrum rows.
// warm / warm_store: see the kernel (a ray of an idle segment reads but does not store).
template <typename T, int S, int LPR, bool ISO>
__device__ __forceinline__ void ray_sweeps(const T (&a)[S], const T (&b)[S],
                                           const T (&su)[S], const T (&sd)[S],
                                           T F_top, T piB_int, int n_sweeps, double wq,
                                           double wg, int sl, bool base_odd, int j_top,
                                           bool want_spec, double* __restrict__ acc,
                                           T* __restrict__ warm, bool warm_store)
{
    using R = AccRows<RayShape<S, LPR, ISO>::NACC, false>;
    ScanF<T, LPR> F;
    scan_factors<T, S, LPR>(a, sl, F);
    T Y[S];
#pragma unroll
    for (int j = 0; j < S; ++j) Y[j] = T(0);
    T fu0 = T(0), fd0 = T(0), o0 = T(0);
    if (warm) {
        // warm start ("still known" from the previous time step): `warm` points at this
        // ray's F_up at the levels 0 .. LPR S, left there by the previous evaluation
        const int base = sl * S;
        o0 = warm[base];
#pragma unroll
        for (int j = 0; j < S; ++j) Y[j] = warm[base + j + 1];
        for (int sw = 1; sw < n_sweeps; ++sw)
            ray_pass<T, S, LPR, ISO, false, false>(a, b, su, sd, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
        ray_pass<T, S, LPR, ISO, false, true>(a, b, su, sd, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
        if (warm_store) {
#pragma unroll
            for (int j = 0; j < S; ++j) warm[base + j + 1] = Y[j];
            if (sl == 0) warm[0] = fu0;
        }
    } else if (n_sweeps == 1) {
        ray_pass<T, S, LPR, ISO, true, true>(a, b, su, sd, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
    } else {
        ray_pass<T, S, LPR, ISO, true, false>(a, b, su, sd, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
        for (int sw = 2; sw < n_sweeps; ++sw)
            ray_pass<T, S, LPR, ISO, false, false>(a, b, su, sd, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
        ray_pass<T, S, LPR, ISO, false, true>(a, b, su, sd, F, Y, o0, fu0, fd0, F_top, piB_int, wq, sl, base_odd, acc);
    }
    if (want_spec) {
        T ft = T(0);
#pragma unroll
        for (int j = 0; j < S; ++j) ft = (j == j_top) ? Y[j] : ft;
        acc[32 * R::SPU] = fma(wg, (double)ft, acc[32 * R::SPU]);
        acc[32 * R::SPD] = fma(wg, (double)fd0, acc[32 * R::SPD]);
    }
}

// ---------------------------------------------------------------------------------------------
// Direct solve (n_scat = HELIOS_NSCAT_DIRECT, reading S12): the n_scat -> infinity
// limit of the sweeps of PAPER.md:292, i.e. the solution of the coupled system of all sublayer relations
// and the two boundary conditions, in O(n) per ray.
//
// A stack of sublayers between a bottom and a top level acts on the fluxes entering it as
//   F_up[top] = t F_up[bot] + rt F_dn[top] + su,     F_dn[bot] = t F_dn[top] + rb F_up[bot] + sd
// (one sublayer: t = a, rt = rb = rho = -beta/alpha).  Stacking X2 on top of X1 is the adding method
// (associative, so it can be scanned over the lanes):
//   d = 1/(1 - rt1 rb2),  t = t1 t2 d,  rt = rt2 + t2^2 d rt1,  rb = rb1 + t1^2 d rb2,
//   su = su2 + t2 d (su1 + rt1 sd2),  sd = sd1 + t1 d (sd2 + rb2 su1).
// 1 - rt1 rb2 loses all digits for thick, nearly conservative stacks (rt, rb -> 1), so a stack is held by
// its transmittance and its two ABSORPTANCES wt = 1 - rt - t, wb = 1 - rb - t (>= 0; zero for eq. 14), in
// which every sum has terms of one sign:
//   1 - rt1 rb2 = (t1 + wt1) rb2 + (t2 + wb2),
//   wt = wt2 + t2 d (wt1 + wb2 rt1),   wb = wb1 + t1 d (wb2 + wt1 rb2).
// The BOA condition (eq. 22) is the stack (t, wt, wb, su, sd) = (0, 0, 1, pi B_int, 0) below level 0.
//   (1) every lane stacks its S sublayers (lane 0 on top of the BOA element);
//   (2) Kogge-Stone scan over the lanes: lane L then holds the stack BOA .. top of lane L, whose
//       c = t + wt = 1 - rt and su = U give F_up = (1 - c) F_dn + U at that level;
//   (3) with (c, U) at its lowest level each lane eliminates upwards through its sublayers (a, w, rho = 1 - a - w):
//         F_dn[s] = e F_dn[s+1] + f,  e = a d,  f = (sd + rho U) d,  d = 1/((a + w) + rho c),
//         c' = w + e (c (1 - w) + w),  U' = a ((1 - c) f + U) + su;
//   (4) F_dn follows from the top (eq. 20) by the affine scan used for the sweeps, F_up = (1 - c) F_dn + U.
template <typename T> __device__ __forceinline__ T rcp_r(T x);
template <> __device__ __forceinline__ double rcp_r<double>(double x) { return rcp_fast(x); }
template <> __device__ __forceinline__ float rcp_r<float>(float x)
{
    float r = rcp_approx(x);
    return fmaf(r, fmaf(-x, r, 1.0f), r);
}

template <typename T>
struct Stack { T t, wt, wb, su, sd; };

// X2 on top of X1
template <typename T>
__device__ __forceinline__ Stack<T> stack_on(const Stack<T>& x1, const Stack<T>& x2)
{
    const T rt1 = (T(1) - x1.t) - x1.wt, rb2 = (T(1) - x2.t) - x2.wb;
    const T d = rcp_r<T>(fma(x1.t + x1.wt, rb2, x2.t + x2.wb));
    const T g2 = x2.t * d, g1 = x1.t * d;
    Stack<T> r;
    r.t = x1.t * g2;
    r.wt = fma(g2, fma(x2.wb, rt1, x1.wt), x2.wt);
    r.wb = fma(g1, fma(x1.wt, rb2, x2.wb), x1.wb);
    r.su = fma(g2, fma(rt1, x2.sd, x1.su), x2.su);
    r.sd = fma(g1, fma(rb2, x1.su, x2.sd), x1.sd);
    return r;
}

// Adds the weighted interface fluxes of the final pass to the lane's accumulator column:
// Yd[j] = F_dn at local level j, Yu[j] = F_up at local level j+1.
template <typename T, int S, int LPR, bool ISO>
__device__ __forceinline__ void ray_accumulate(const T (&Yd)[S], const T (&Yu)[S], T fu0, T F_top, double wq,
                                               bool base_odd, double* __restrict__ acc)
{
    constexpr int NACC = RayShape<S, LPR, ISO>::NACC;
    using R = AccRows<NACC, false>;
#pragma unroll
    for (int k = 0; k < NACC; ++k) {
        T vd, vu;
        if (ISO) { vd = Yd[k]; vu = Yu[k]; }
        else {
            const T de = Yd[(2 * k < S) ? 2 * k : 0];
            const T dodd = (2 * k + 1 < S) ? Yd[(2 * k + 1 < S) ? 2 * k + 1 : 0] : T(0);
            vd = base_odd ? dodd : de;
            const T ue = (2 * k + 1 < S) ? Yu[(2 * k + 1 < S) ? 2 * k + 1 : 0] : T(0);
            const T uo = Yu[(2 * k < S) ? 2 * k : 0];
            vu = base_odd ? uo : ue;
        }
        acc[32 * (R::DN + k)] = fma(wq, (double)vd, acc[32 * (R::DN + k)]);
        acc[32 * (R::UP + k)] = fma(wq, (double)vu, acc[32 * (R::UP + k)]);
    }
    acc[32 * R::UP0] = fma(wq, (double)fu0, acc[32 * R::UP0]);
    acc[32 * R::DNT] = fma(wq, (double)F_top, acc[32 * R::DNT]);
}

template <typename T, int S, int LPR, bool ISO>
__device__ __forceinline__ void ray_direct(T (&a)[S], T (&b)[S], T (&su)[S], T (&sd)[S],
                                           T F_top, T piB_int, double wq, double wg, int sl,
                                           bool base_odd, int j_top, bool want_spec,
                                           double* __restrict__ acc)
{
    using R = AccRows<RayShape<S, LPR, ISO>::NACC, false>;
    constexpr int NR = SegOf<LPR>::ROUNDS;
    // (1) the lane's stack; sub-lane 0 starts from the BOA element, the others from the empty stack.
    //     b[] holds the absorptances w (ray_coefficients<..., WABS = true>).
    Stack<T> X;
    X.t = (sl == 0) ? T(0) : T(1);
    X.wt = T(0);
    X.wb = (sl == 0) ? T(1) : T(0);
    X.su = (sl == 0) ? piB_int : T(0);
    X.sd = T(0);
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const T w = b[j], rho = (T(1) - a[j]) - w;
        const T rt1 = (T(1) - X.t) - X.wt;
        const T d = rcp_r<T>(fma(X.t + X.wt, rho, a[j] + w));
        const T g2 = a[j] * d, g1 = X.t * d;
        const T su_n = fma(g2, fma(rt1, sd[j], X.su), su[j]);
        const T sd_n = fma(g1, fma(rho, X.su, sd[j]), X.sd);
        const T wt_n = fma(g2, fma(w, rt1, X.wt), w);
        X.wb = fma(g1, fma(X.wt, rho, w), X.wb);
        X.wt = wt_n;
        X.t = X.t * g2;
        X.su = su_n;
        X.sd = sd_n;
    }
    // (2) inclusive scan over the lanes of the ray (lower lanes = lower stacks)
#pragma unroll
    for (int k = 0; k < NR; ++k) {
        const int dd = 1 << k;
        Stack<T> lo;
        lo.t = shfl_up_w<LPR>(X.t, dd);
        lo.wt = shfl_up_w<LPR>(X.wt, dd);
        lo.wb = shfl_up_w<LPR>(X.wb, dd);
        lo.su = shfl_up_w<LPR>(X.su, dd);
        lo.sd = shfl_up_w<LPR>(X.sd, dd);
        const Stack<T> c = stack_on(lo, X);
        const bool has = sl >= dd;
        X.t = has ? c.t : X.t;
        X.wt = has ? c.wt : X.wt;
        X.wb = has ? c.wb : X.wb;
        X.su = has ? c.su : X.su;
        X.sd = has ? c.sd : X.sd;
    }
    // (c, U) at this lane's local level 0 = top of the stack held by the lane below
    T cv = shfl_up_w<LPR>(X.t + X.wt, 1), Uv = shfl_up_w<LPR>(X.su, 1);
    cv = (sl == 0) ? T(0) : cv;
    Uv = (sl == 0) ? piB_int : Uv;
    // (3) eliminate upwards: a <- e, sd <- f, b <- c, su <- U at local level j
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const T w = b[j], rho = (T(1) - a[j]) - w;
        const T d = rcp_r<T>(fma(rho, cv, a[j] + w));
        const T e = a[j] * d;
        const T f = fma(rho, Uv, sd[j]) * d;
        const T cn = fma(e, fma(cv, T(1) - w, w), w);
        const T Un = fma(a[j], fma(T(1) - cv, f, Uv), su[j]);
        a[j] = e;
        sd[j] = f;
        b[j] = cv;
        su[j] = Uv;
        cv = cn;
        Uv = Un;
    }
    // (4) F_dn from the top: affine scan of F_dn[s] = e F_dn[s+1] + f over the lanes
    T Yd[S], Yu[S];
    T run = T(0), AL = T(1);
#pragma unroll
    for (int j = S - 1; j >= 0; --j) {
        run = fma(a[j], run, sd[j]);
        AL *= a[j];
    }
    T C = run, td = AL;
#pragma unroll
    for (int k = 0; k < NR; ++k) {
        const int dd = 1 << k;
        const bool has = sl + dd < LPR;
        const T oc = shfl_down_w<LPR>(C, dd), od = shfl_down_w<LPR>(td, dd);
        C = has ? fma(td, oc, C) : C;
        td = has ? td * od : td;
    }
    const T out = fma(td, F_top, C);                         // F_dn at this lane's local level 0
    T q = shfl_down_w<LPR>(out, 1);
    q = (sl == LPR - 1) ? F_top : q;                         // F_dn at local level S (eq. 20 above the top lane)
    Yd[S - 1] = fma(a[S - 1], q, sd[S - 1]);
#pragma unroll
    for (int j = S - 2; j >= 0; --j) Yd[j] = fma(a[j], Yd[j + 1], sd[j]);
#pragma unroll
    for (int j = 0; j + 1 < S; ++j) Yu[j] = fma(-b[j + 1], Yd[j + 1], Yd[j + 1] + su[j + 1]);   // F_up at local level j+1
    Yu[S - 1] = fma(-cv, q, q + Uv);
    const T fd0 = shfl_idx_w<LPR>(Yd[0], 0);
    const T fu0 = fd0 + piB_int;                             // eq. 22
    ray_accumulate<T, S, LPR, ISO>(Yd, Yu, fu0, F_top, wq, base_odd, acc);
    if (want_spec) {
        T ft = T(0);
#pragma unroll
        for (int j = 0; j < S; ++j) ft = (j == j_top) ? Yu[j] : ft;
        acc[32 * R::SPU] = fma(wg, (double)ft, acc[32 * R::SPU]);
        acc[32 * R::SPD] = fma(wg, (double)fd0, acc[32 * R::SPD]);
    }
}

}  // namespace hx
