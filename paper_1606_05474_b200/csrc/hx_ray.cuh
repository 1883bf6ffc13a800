// hx_ray.cuh -- one ray (column, bin, g) of the two-stream solve held in the registers of one warp.
// Product code (CUDA path); shares nothing with oracle/.
//
// Layout.  The padded column has 32*S sublayers; lane L owns sublayers L*S .. L*S+S-1 ("local"
// j = 0..S-1) and the levels L*S .. L*S+S-1; level L*S+S is the next lane's local level 0.
// Padded sublayers have dtau = 0, for which the coefficients below reduce to the identity map,
// so the TOA boundary value simply travels through them.
//
// Per sublayer (eq. 8, 11-15 with readings G1, G2, G5, S2 of DESIGN.md):
//   F_dn[s]   = a F_dn[s+1] - b F_up[s]   + sd        a = xi/alpha, b = beta/alpha,
//   F_up[s+1] = a F_up[s]   - b F_dn[s+1] + su        sd = S_dn/alpha, su = S_up/alpha
// With the other direction's fluxes frozen, one sweep is an affine recurrence along the column.
// Each lane runs it over its S sublayers from a zero input (which yields the lane's affine map
// (A, C)), the 32 maps are combined by a Kogge-Stone scan with warp shuffles, and the lane's true
// input is then added back: F[j] += (prod of a down to j) * F_in.  A's partial products do not
// depend on the sweep and are formed once per ray.
#pragma once
#include "helios_internal.h"
#include "hx_math.cuh"

namespace hx {

constexpr unsigned kFull = 0xffffffffu;

template <int S, bool ISO>
struct RayShape {
    static constexpr int NSUB_PAD = 32 * S;
    static constexpr int NN = NSUB_PAD + 1;                 // node slots (levels) incl. the top one
    static constexpr int KLS = ((NN + 7) & ~15) + 8;        // kappa stage row stride (== 8 mod 16)
    static constexpr int UP = ISO ? 0 : 1;                  // node offset of a sublayer's upper end
    static constexpr int NACC = ISO ? S : (S + 1) / 2;      // interface accumulators per lane
};

// Accumulators a warp carries over all its (bin, g) rays.
template <int NACC>
struct RayAcc {
    double up[NACC];   // sum w dnu F_up at the lane's interface levels (up-sweep ownership)
    double dn[NACC];   // sum w dnu F_dn at the lane's interface levels (down-sweep ownership)
    double up0;        // F_up at level 0 (BOA); meaningful on every lane, lane 0 writes it
    double dnT;        // F_dn at level 32*S (the boundary value itself); lane 31 writes it
};

// Sublayer coefficients for the lane's S sublayers.  kap/Bn point at the lane's first node.
template <int S, bool ISO>
__device__ __forceinline__ void ray_coefficients(const BinConst& bc, double tpe, double dtau_iso,
                                                 const double* __restrict__ kap,
                                                 const double* __restrict__ hP,
                                                 const double* __restrict__ Bn,
                                                 double (&a)[S], double (&b)[S], double (&su)[S],
                                                 double (&sd)[S])
{
    constexpr int UP = RayShape<S, ISO>::UP;
    double k_lo = kap[0], B_lo = Bn[0];
#pragma unroll
    for (int j = 0; j < S; ++j) {
        const double k_up = ISO ? k_lo : kap[j + 1];
        const double B_up = ISO ? B_lo : Bn[j + 1];
        const double dtau = hP[j] * (k_lo + k_up);                   // eq. 19, kappa = mean of the ends
        if (!bc.pure_scat) {
            const double tr = exp2_nonpos(bc.nlam2 * dtau);         // eq. 8
            const double tr2 = tr * tr;
            const double alpha = fma(bc.zm2, tr2, -bc.zp2);         // eq. 12
            const double beta = bc.zpzm * fma(-tr, tr, 1.0);
            const double xi = -bc.r * tr;                           // (zm^2 - zp^2) T = -r T
            const bool thin = !(dtau >= dtau_iso) || !(dtau > 0.0);
            const double dsafe = thin ? 1.0 : dtau;
            const double inv = 1.0 / (alpha * dsafe);               // one reciprocal for 1/alpha, 1/dtau
            const double ia = dsafe * inv;
            const double apb = alpha + beta;
            // eq. 15 (G1: destination-side B with (alpha+beta), source-side B with xi)
            const double Bp = (B_lo - B_up) * (alpha * inv);        // eq. 5, dB/dtau
            const double t = bc.kp * Bp * (alpha - xi - beta);
            double s_up = fma(B_up, apb, fma(-B_lo, xi, t));
            double s_dn = fma(B_lo, apb, fma(-B_up, xi, -t));
            // eq. 11 with beta - v == alpha + beta - xi (G5) and B = mean of the ends (S2)
            const double s_iso = 0.5 * (B_lo + B_up) * (apb - xi);
            s_up = thin ? s_iso : s_up;
            s_dn = thin ? s_iso : s_dn;
            const double f = tpe * ia;
            a[j] = xi * ia;
            b[j] = beta * ia;
            su[j] = s_up * f;
            sd[j] = s_dn * f;
        } else {                                                    // eq. 14
            const double x = bc.xfac * dtau;
            const double inv = 1.0 / (2.0 + x);
            a[j] = 2.0 * inv;
            b[j] = -x * inv;
            su[j] = 0.0;
            sd[j] = 0.0;
        }
        if (!ISO) { k_lo = k_up; B_lo = B_up; }
        else if (j + 1 < S) { k_lo = kap[j + 1]; B_lo = Bn[j + 1]; }
    }
}

// Runs n_sweeps x (down sweep, BOA condition, up sweep) for one ray and adds the final sweep's
// interface fluxes, weighted by wq = w_g * dnu, to acc.  Returns through fd_boa / fu_toa the
// final F_dn(level 0) (all lanes) and, on lane lane_top, F_up at the lane's local level j_top+1.
template <int S, bool ISO>
__device__ __forceinline__ void ray_sweeps(const double (&a)[S], const double (&b)[S],
                                           const double (&su)[S], const double (&sd)[S],
                                           double F_top, double piB_int, int n_sweeps, double wq,
                                           int lane, bool base_odd, int j_top,
                                           RayAcc<RayShape<S, ISO>::NACC>& acc,
                                           double& fd_boa, double& fu_toa)
{
    constexpr int NACC = RayShape<S, ISO>::NACC;
    // sweep-independent partial products of the scan
    double Ad[5], Au[5], Ad5, Au5;
    {
        double AL = a[0];
#pragma unroll
        for (int j = 1; j < S; ++j) AL *= a[j];
        double td = AL, tu = AL;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const int d = 1 << k;
            const double od = __shfl_down_sync(kFull, td, d);
            const double ou = __shfl_up_sync(kFull, tu, d);
            Ad[k] = td;
            Au[k] = tu;
            if (lane + d < 32) td *= od;
            if (lane >= d) tu *= ou;
        }
        Ad5 = td;
        Au5 = tu;
    }
    double Y[S];
#pragma unroll
    for (int j = 0; j < S; ++j) Y[j] = 0.0;     // "starting with the coupled dependencies as zero"
    double fu0 = 0.0, fd0 = 0.0;

    for (int sw = 0; sw < n_sweeps; ++sw) {
        // ---- down sweep: Y[j-1] holds F_up at local level j (Y of the lane below for j = 0)
        {
            double o0 = __shfl_up_sync(kFull, Y[S - 1], 1);
            if (lane == 0) o0 = fu0;
            double run = 0.0;
#pragma unroll
            for (int j = S - 1; j >= 0; --j) {
                const double other = (j > 0) ? Y[j > 0 ? j - 1 : 0] : o0;
                const double c = fma(-b[j], other, sd[j]);
                run = fma(a[j], run, c);
                Y[j] = run;
            }
            double C = run;
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const int d = 1 << k;
                const double o = __shfl_down_sync(kFull, C, d);
                if (lane + d < 32) C = fma(Ad[k], o, C);
            }
            const double out = fma(Ad5, F_top, C);              // F_dn at this lane's local level 0
            double q = __shfl_down_sync(kFull, out, 1);
            if (lane == 31) q = F_top;                          // eq. 20 enters above the top lane
#pragma unroll
            for (int j = S - 1; j >= 0; --j) {
                q *= a[j];
                Y[j] += q;
            }
            fd0 = __shfl_sync(kFull, Y[0], 0);
            fu0 = fd0 + piB_int;                                // eq. 22
        }
        const bool last = (sw + 1 == n_sweeps);
        if (last) {
#pragma unroll
            for (int k = 0; k < NACC; ++k) {
                double v;
                if (ISO) v = Y[k];
                else {
                    const double ve = Y[(2 * k < S) ? 2 * k : 0];
                    const double vo = (2 * k + 1 < S) ? Y[(2 * k + 1 < S) ? 2 * k + 1 : 0] : 0.0;
                    v = base_odd ? vo : ve;
                }
                acc.dn[k] = fma(wq, v, acc.dn[k]);
            }
        }
        // ---- up sweep: Y[j+1] holds F_dn at local level j+1 (Y[0] of the lane above for j = S-1)
        {
            double oS = __shfl_down_sync(kFull, Y[0], 1);
            if (lane == 31) oS = F_top;
            double run = 0.0;
#pragma unroll
            for (int j = 0; j < S; ++j) {
                const double other = (j + 1 < S) ? Y[(j + 1 < S) ? j + 1 : 0] : oS;
                const double c = fma(-b[j], other, su[j]);
                run = fma(a[j], run, c);
                Y[j] = run;
            }
            double C = run;
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const int d = 1 << k;
                const double o = __shfl_up_sync(kFull, C, d);
                if (lane >= d) C = fma(Au[k], o, C);
            }
            const double out = fma(Au5, fu0, C);                // F_up at this lane's local level S
            double q = __shfl_up_sync(kFull, out, 1);
            if (lane == 0) q = fu0;
#pragma unroll
            for (int j = 0; j < S; ++j) {
                q *= a[j];
                Y[j] += q;                                      // F_up at local level j+1
            }
        }
        if (last) {
#pragma unroll
            for (int k = 0; k < NACC; ++k) {
                double v;
                if (ISO) v = Y[k];
                else {
                    // level base + j + 1 even: j = 2k+1 for an even base, j = 2k for an odd base
                    const double ve = (2 * k + 1 < S) ? Y[(2 * k + 1 < S) ? 2 * k + 1 : 0] : 0.0;
                    const double vo = Y[(2 * k < S) ? 2 * k : 0];
                    v = base_odd ? vo : ve;
                }
                acc.up[k] = fma(wq, v, acc.up[k]);
            }
            acc.up0 = fma(wq, fu0, acc.up0);
            acc.dnT = fma(wq, F_top, acc.dnT);
        }
    }
    fd_boa = fd0;
    double ft = 0.0;
#pragma unroll
    for (int j = 0; j < S; ++j) ft = (j == j_top) ? Y[j] : ft;
    fu_toa = ft;
}

}  // namespace hx
