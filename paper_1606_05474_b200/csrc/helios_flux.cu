// helios_flux.cu -- the ray kernel: steps a0-a8 of include/helios.h for every (column, bin, g).
// Product code (CUDA path, sm_100a); shares nothing with oracle/.
//
// Grid = (columns, bin chunks); block = `warps` warps working on one column.  A warp owns a run of
// consecutive bins; per bin it
//   (1) evaluates the incomplete Planck integral at the bin's upper edge for every level (lanes over
//       levels; the lower edge is carried from the previous bin) and forms the bin-mean Planck
//       function per level in shared memory (a2),
//   (2) per group of 4 Gauss points interpolates the k-table at every level with lanes running over
//       (level, g) so that the four corner loads are 32-byte contiguous per level (a1), staging
//       kappa in shared memory,
//   (3) runs hx::ray_coefficients / hx::ray_sweeps (a3-a7) for RPW = 32 / LPR Gauss points at a time, each ray
//       in the registers of LPR lanes (lanes over sublayers; hx_ray.cuh), accumulating w_g*dnu*F at the lane's
//       interface levels (a8).
// The block then adds the warps' accumulators in a fixed order and writes one partial sum (a double-double
// pair) per (chunk, column); k_reduce (helios_aux.cu) adds the chunks in order.  No atomics: bit-reproducible.
//
// This file is compiled once per UNIT = (variant HX_FLUX_ALT, arithmetic HX_FLUX_F32, lanes per ray HX_FLUX_LPR)
// by build.py, in parallel.  Variants: 0 = the two-stream kernel (sweeps of PAPER.md:292 or the direct coupled
// solve, S12), the one the benchmark times; 1 = the same plus the exact pure-absorption limit (S13,
// whose E_1 evaluation is a real function call) and the albedo-per-sublayer coefficients of
// helios_set_scattering (S14); 2 = variant 0 plus the tabulated Planck function (S15).  They are separate
// kernels because each extra path costs the sweeps registers (round 1: +2.2 % / +0.75 % time when merged).
#ifndef HX_FLUX_ALT
#define HX_FLUX_ALT 0
#endif
#ifndef HX_FLUX_F32
#define HX_FLUX_F32 0
#endif
#ifndef HX_FLUX_LPR
#define HX_FLUX_LPR 16
#endif
#include "helios_internal.h"
#include "hx_math.cuh"
#include "hx_ray.cuh"

// HX_CHECKED (build.py --checked; developer builds): the kernel's own memory checker, used where compute-sanitizer
// is not available.  (1) all dynamic shared memory starts as NaN patterns, and the kappa stage (which doubles as the
// Planck stage) is re-poisoned whenever its content is dead, so a read of something not (re)written shows up as NaN
// in the fluxes; (2) guard words behind the block region and every warp region are verified at the end; (3) every
// index formed from run-time values is checked.  A failure sets flags[3] to a code that the host calls report.
#ifdef HX_CHECKED
#define HX_CHECK(cond, code) do { if (!(cond)) atomicMax(v.check_fail, (int32_t)(code)); } while (0)
constexpr int kGuardBytes = 16;
#else
#define HX_CHECK(cond, code) ((void)0)
constexpr int kGuardBytes = 0;
#endif

#define HX_CAT4_(a, b, c, d) a##b##c##d
#define HX_CAT4(a, b, c, d) HX_CAT4_(a, b, c, d)
#if HX_FLUX_ALT == 1
#define HX_ALT_TAG _alt
#elif HX_FLUX_ALT == 2
#define HX_ALT_TAG _tab
#else
#define HX_ALT_TAG _main
#endif
#if HX_FLUX_F32
#define HX_PREC_TAG _f32
#else
#define HX_PREC_TAG _f64
#endif
#if HX_FLUX_LPR == 8
#define HX_LPR_TAG _l8
#elif HX_FLUX_LPR == 16
#define HX_LPR_TAG _l16
#else
#define HX_LPR_TAG _l32
#endif
#define HX_UNIT_NAME(base) HX_CAT4(base, HX_ALT_TAG, HX_PREC_TAG, HX_LPR_TAG)

namespace hx {

// Everything of this unit lives in a namespace named after the unit.  NOT an anonymous namespace: nvcc gives the
// entities of an anonymous namespace weak symbols under a prefix derived from the source FILE, so the host-side
// templates (launch_one<13, 16, false, float>, the kernel stubs) of the 18 units compiled from this file would
// be merged by the linker and every variant would launch the first unit's kernel.
namespace HX_UNIT_NAME(unit) {

// Row stride of the kappa stage (elements; one row per Gauss point of the staged group).
// fp64: == 4 mod 8 -- the staging stores rows 0 and 2 (1 and 3) from the two lanes of a pair, and rows two apart
// then lie 16 banks apart (measured against == 8 mod 16: -0.75 % time); the coefficient stage reads one row per
// ray with stride S, one half-warp per 64-bit access.  fp32: all 32 lanes of a read are served together, ray r of
// the warp reading row r with lane stride S: the stride (a multiple of 4) with the fewest lanes per bank.
template <int S, int LPR, int NN, int BYTES>
constexpr int stage_stride()
{
    if (BYTES == 8) return ((NN + 7) & ~7) + 4;
    int best = 0, best_cost = 1 << 30;
    for (int k = (NN + 3) & ~3; k < ((NN + 3) & ~3) + 32; k += 4) {
        int cnt[32] = {}, cost = 0;
        for (int lane = 0; lane < 32; ++lane) {
            const int c = ++cnt[((lane / LPR) * k + (lane % LPR) * S) & 31];
            cost = c > cost ? c : cost;
        }
        if (cost < best_cost) { best_cost = cost; best = k; }
    }
    return best;
}

// Shared-memory carve-up (byte offsets).  Real = double (fp64 path) or float (fp32 ray arithmetic; the
// Planck integrals, node temperatures and all accumulators stay fp64).
template <int S, int LPR, bool ISO, typename Real>
struct Smem {
    using Sh = RayShape<S, LPR, ISO>;
    static constexpr bool COMP = sizeof(Real) == 8;
    static constexpr int NPL = (Sh::NN + 31) / 32;                           // nodes per lane (lanes over nodes)
    static constexpr int al(int x) { return (x + 15) & ~15; }
    static constexpr int KLS = stage_stride<S, LPR, Sh::NN, (int)sizeof(Real)>();     // kappa stage row stride
    static constexpr int W4 = 0;                                             // Real[NN][4] bilinear weights * kscale
    static constexpr int TN = al(W4 + (int)sizeof(Real) * 4 * Sh::NN);       // double[NN] node temperatures
    static constexpr int TI = al(TN + 8 * Sh::NN);                           // double[NN] 1/T
    static constexpr int HP = al(TI + 8 * Sh::NN);                           // Real[LPR S] (P_lo-P_up)/(2g)
    static constexpr int NOFF = al(HP + (int)sizeof(Real) * Sh::NSUB_PAD);   // int32[NN] table offsets
    static constexpr int ETAB = al(NOFF + 4 * Sh::NN);                       // double[256] 2^(j/256)
    static constexpr int BLOCK = al(ETAB + 8 * kExpTab + kGuardBytes);
    static constexpr int W_KST = 0;                                          // per warp: Real[4][KLS] kappa stage
    static constexpr int W_B = al(W_KST + (int)sizeof(Real) * kGroupG * KLS);   // Real[2][LPR S] (2 pi/D) * (mean, half difference) of the bin-mean Planck function over a sublayer
    static constexpr int W_G = al(W_B + (int)sizeof(Real) * 2 * Sh::NSUB_PAD);      // double[NPL][32] Planck edge values
    static constexpr int W_ACC = al(W_G + 8 * 32 * NPL);                     // double[ROWS][32] accumulators
    static constexpr int WARP = al(W_ACC + 8 * 32 * AccRows<Sh::NACC, COMP>::ROWS + kGuardBytes);
    static __host__ __device__ size_t bytes(int warps) { return (size_t)BLOCK + (size_t)warps * WARP; }
};

// Planck edge values (-H(x) for x < kPlanckSwitch, G(x) above; x = xe/T) for the NJ nodes lane + 32 j of this lane;
// invT points at the lane's first node (stride 32), out[NJ] is the caller's register array.  Nodes at or
// beyond n_act are skipped (their out value is meaningless).
template <int NJ>
__device__ __forceinline__ void planck_edges(double xe, const double* __restrict__ invT, int lane, int n_act,
                                             double (&out)[NJ])
{
    double x[NJ], e1[NJ], em[NJ], sum[NJ];
    int M = 0;
    bool any_low = false;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        const bool act = lane + 32 * j < n_act;
        x[j] = xe * (act ? invT[32 * j] : 1.0);
        e1[j] = exp_nonpos(-x[j]);
        em[j] = 1.0;
        sum[j] = 0.0;
        if (act && x[j] >= kPlanckSwitch) M = max(M, planck_upper_terms(x[j]));
        if (act && x[j] < kPlanckSwitch) any_low = true;
    }
    M = __reduce_max_sync(kFull, M);
    for (int m = 1; m <= M; ++m) {
        const double rm = c_inv_m[m];
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            em[j] *= e1[j];
            sum[j] += planck_upper_term(x[j], x[j] * x[j], x[j] * x[j] * x[j], em[j], rm);
        }
    }
    if (__any_sync(kFull, any_low)) {
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (x[j] < kPlanckSwitch) sum[j] = -planck_lower(x[j]);
    }
#pragma unroll
    for (int j = 0; j < NJ; ++j) out[j] = sum[j];
}

// k-table staging for one group of 4 Gauss points (a1), fp64: lanes run over (node, g pair) with
// 16-byte loads, KB nodes per lane in flight; scalar fallback for odd n_g / unaligned tables.
template <int NN, int KLS>
__device__ __forceinline__ void stage_kappa(const DevView& v, const double* __restrict__ w4,
                                            const int32_t* __restrict__ noff, double* __restrict__ kst,
                                            int bin, int g0, int lane, size_t sT, size_t sP)
{
    const bool vec2 = ((v.ng & 1) == 0) && ((reinterpret_cast<uintptr_t>(v.ktab) & 15) == 0);
    if (vec2) {
        constexpr int KB = 7;     // nodes per lane in flight (the ray registers are free here): 3 -> 7: -0.3 % time
        // lanes (2s, 2s+1) load the two g pairs of node s: a quarter-warp's 16-byte loads cover whole 32-byte sectors
        // (measured: the pair on the lane's high bit instead -- conflict-free stores -- costs 4.4 % of the kernel)
        const int pr = lane & 1;
        const int g = min(g0 + 2 * pr, v.ng - 2);
        const double* __restrict__ pb = v.ktab + (size_t)bin * v.ng + g;
        double* __restrict__ krow = kst + (2 * pr) * KLS;
        for (int s0 = lane >> 1; s0 < NN; s0 += 16 * KB) {
            double2 k00[KB], k01[KB], k10[KB], k11[KB];
#pragma unroll
            for (int u = 0; u < KB; ++u) {
                const int s = min(s0 + 16 * u, NN - 1);
                const double* __restrict__ p = pb + (size_t)noff[s];
                k00[u] = __ldg(reinterpret_cast<const double2*>(p));
                k01[u] = __ldg(reinterpret_cast<const double2*>(p + sT));
                k10[u] = __ldg(reinterpret_cast<const double2*>(p + sP));
                k11[u] = __ldg(reinterpret_cast<const double2*>(p + sP + sT));
            }
#pragma unroll
            for (int u = 0; u < KB; ++u) {
                const int s = s0 + 16 * u;
                if (s < NN) {
                    const double2 wa = *reinterpret_cast<const double2*>(w4 + 4 * s);
                    const double2 wb = *reinterpret_cast<const double2*>(w4 + 4 * s + 2);
                    krow[s] = fma(wa.x, k00[u].x, fma(wa.y, k01[u].x, fma(wb.x, k10[u].x, wb.y * k11[u].x)));
                    krow[KLS + s] = fma(wa.x, k00[u].y, fma(wa.y, k01[u].y, fma(wb.x, k10[u].y, wb.y * k11[u].y)));
                }
            }
        }
    } else {
        for (int idx = lane; idx < NN * kGroupG; idx += 32) {
            const int s = idx >> 2, gg = idx & 3;
            const int g = min(g0 + gg, v.ng - 1);
            const double* __restrict__ p = v.ktab + (size_t)noff[s] + (size_t)bin * v.ng + g;
            const double2 wa = *reinterpret_cast<const double2*>(w4 + 4 * s);
            const double2 wb = *reinterpret_cast<const double2*>(w4 + 4 * s + 2);
            const double k00 = __ldg(p), k01 = __ldg(p + sT), k10 = __ldg(p + sP), k11 = __ldg(p + sP + sT);
            kst[gg * KLS + s] = fma(wa.x, k00, fma(wa.y, k01, fma(wb.x, k10, wb.y * k11)));
        }
    }
}

// fp32: the table was converted to float at set-up (v.ktab32); lanes run over nodes and load the
// four Gauss points of the group as one float4 per corner.
template <int NN, int KLS>
__device__ __forceinline__ void stage_kappa(const DevView& v, const float* __restrict__ w4,
                                            const int32_t* __restrict__ noff, float* __restrict__ kst,
                                            int bin, int g0, int lane, size_t sT, size_t sP)
{
    const bool vec4 = ((v.ng & 3) == 0);
    if (vec4) {
        // nodes per lane in flight: all of them in one round when the column allows it (the ray registers are free
        // here; 100 layers: 7 x 4 float4).  Measured on config 4: 2 -> 7: -2.5 % time, 4 (two uneven rounds): +3 %.
        constexpr int KB = (NN + 31) / 32 < 7 ? (NN + 31) / 32 : 7;
        const float* __restrict__ pb = v.ktab32 + (size_t)bin * v.ng + g0;
        for (int s0 = lane; s0 < NN; s0 += 32 * KB) {
            float4 k00[KB], k01[KB], k10[KB], k11[KB];
#pragma unroll
            for (int u = 0; u < KB; ++u) {
                const int s = min(s0 + 32 * u, NN - 1);
                const float* __restrict__ p = pb + (size_t)noff[s];
                k00[u] = __ldg(reinterpret_cast<const float4*>(p));
                k01[u] = __ldg(reinterpret_cast<const float4*>(p + sT));
                k10[u] = __ldg(reinterpret_cast<const float4*>(p + sP));
                k11[u] = __ldg(reinterpret_cast<const float4*>(p + sP + sT));
            }
#pragma unroll
            for (int u = 0; u < KB; ++u) {
                const int s = s0 + 32 * u;
                if (s < NN) {
                    const float4 w = *reinterpret_cast<const float4*>(w4 + 4 * s);
                    kst[s] = fmaf(w.x, k00[u].x, fmaf(w.y, k01[u].x, fmaf(w.z, k10[u].x, w.w * k11[u].x)));
                    kst[KLS + s] = fmaf(w.x, k00[u].y, fmaf(w.y, k01[u].y, fmaf(w.z, k10[u].y, w.w * k11[u].y)));
                    kst[2 * KLS + s] = fmaf(w.x, k00[u].z, fmaf(w.y, k01[u].z, fmaf(w.z, k10[u].z, w.w * k11[u].z)));
                    kst[3 * KLS + s] = fmaf(w.x, k00[u].w, fmaf(w.y, k01[u].w, fmaf(w.z, k10[u].w, w.w * k11[u].w)));
                }
            }
        }
    } else {
        for (int idx = lane; idx < NN * kGroupG; idx += 32) {
            const int s = idx >> 2, gg = idx & 3;
            const int g = min(g0 + gg, v.ng - 1);
            const float* __restrict__ p = v.ktab32 + (size_t)noff[s] + (size_t)bin * v.ng + g;
            const float4 w = *reinterpret_cast<const float4*>(w4 + 4 * s);
            kst[gg * KLS + s] = fmaf(w.x, __ldg(p), fmaf(w.y, __ldg(p + sT), fmaf(w.z, __ldg(p + sP), w.w * __ldg(p + sP + sT))));
        }
    }
}

// VARIANT = HX_FLUX_ALT is a template parameter so that a profiler's kernel list tells the variants apart.
template <int VARIANT, int S, int LPR, bool ISO, typename Real>
__global__ void __launch_bounds__(32 * FluxWarps<S, sizeof(Real) == 4>::value, 1)
k_flux(const DevView v, const int respect_converged)
{
    static_assert(VARIANT == HX_FLUX_ALT, "one variant per translation unit");
    using Sh = RayShape<S, LPR, ISO>;
    using Sm = Smem<S, LPR, ISO, Real>;
    constexpr int NN = Sh::NN, KLS = Sm::KLS, NACC = Sh::NACC, NPL = Sm::NPL, RPW = SegOf<LPR>::RPW;
    constexpr int NSL = (Sh::NSUB_PAD + 31) / 32;         // sublayers per lane when lanes run over sublayers
    constexpr bool F32 = sizeof(Real) == 4;
    constexpr bool COMP = Sm::COMP;
    static_assert(kGroupG % RPW == 0, "a staged group of Gauss points holds whole sets of rays");
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int c = blockIdx.x, chunk = blockIdx.y;      // column-fastest dispatch within a bin chunk
    if (respect_converged && (v.converged[c] || v.col_nonfinite[c])) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const int sl = lane & (LPR - 1), rw = lane / LPR;  // sub-lane within the ray, ray within the warp

    Real* w4 = reinterpret_cast<Real*>(smem_raw + Sm::W4);
    double* Tn = reinterpret_cast<double*>(smem_raw + Sm::TN);
    double* Ti = reinterpret_cast<double*>(smem_raw + Sm::TI);
    Real* hPs = reinterpret_cast<Real*>(smem_raw + Sm::HP);
    int32_t* noff = reinterpret_cast<int32_t*>(smem_raw + Sm::NOFF);
    double* exp_tab = reinterpret_cast<double*>(smem_raw + Sm::ETAB);
    unsigned char* wsm = smem_raw + Sm::BLOCK + (size_t)warp * Sm::WARP;
    Real* kst = reinterpret_cast<Real*>(wsm + Sm::W_KST);
    Real* Bw = kst;                                   // per-node Planck values of the bin: the kappa stage is idle then
    Real* Bmw = reinterpret_cast<Real*>(wsm + Sm::W_B);
    Real* Bhw = Bmw + Sh::NSUB_PAD;
    double* Gw = reinterpret_cast<double*>(wsm + Sm::W_G) + lane;      // this lane's Planck edge values, stride 32
    double* accw = reinterpret_cast<double*>(wsm + Sm::W_ACC);
    double* acc = accw + lane;                        // this lane's accumulator column, row stride 32
    // [warps][2][bin id, up, down] spectrum shares of the partial bins at the ends of a warp's unit run (unit_split
    // plans only), after the per-warp regions
    double* specbuf = reinterpret_cast<double*>(smem_raw + Sm::BLOCK + (size_t)(blockDim.x >> 5) * Sm::WARP);

#ifdef HX_CHECKED
    {
        const size_t total = Sm::bytes(blockDim.x >> 5) + (v.unit_split ? (size_t)(blockDim.x >> 5) * 48 : 0);
        for (size_t i = tid; i < total / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(smem_raw)[i] = 0xFFFFFFFFu;   // NaN
        __syncthreads();
        if (tid == 0) *reinterpret_cast<unsigned long long*>(smem_raw + Sm::BLOCK - 8) = 0x600DC0DE600DC0DEull;
        if (lane == 0) *reinterpret_cast<unsigned long long*>(wsm + Sm::WARP - 8) = 0x600DC0DE600DC0DEull;
        __syncthreads();
    }
#endif
    // ---- a0 + table cell / weights of every node (block prologue)
    const double* __restrict__ Tc = v.T + (size_t)c * v.n;
    const double ksc = v.kscale[c];
    const int n = v.n, nnode = v.nnode;
    const double tab_t0 = v.tab_axis[0], tab_inv_dt = v.tab_axis[1];
    for (int s = tid; s < NN; s += blockDim.x) {
        const int node = min(s, nnode - 1);        // slots beyond the column repeat its last node (their sublayers have dtau = 0)
        double T;
        if (ISO) {
            T = Tc[node];
        } else if (node & 1) {
            T = Tc[node >> 1];
        } else {                                   // interface j: linear in log P
            const int j = node >> 1;
            if (n == 1) T = Tc[0];
            else {
                int ia = j - 1, ib = j;
                if (j == 0) { ia = 0; ib = 1; }
                if (j == n) { ia = n - 2; ib = n - 1; }
                T = fma(v.w_iface[j], Tc[ib] - Tc[ia], Tc[ia]);
                T = fmax(T, 1.0);
            }
        }
        Tn[s] = T;
        Ti[s] = 1.0 / T;
        double tt = (T - tab_t0) * tab_inv_dt;          // PAPER.md:376, 398 (clamped, fn. 9)
        tt = fmin(fmax(tt, 0.0), (double)(v.ntab_t - 1));
        const int it = min((int)tt, v.ntab_t - 2);
        const double ft = tt - (double)it;
        const int ip = v.node_ip[node];
        const double fp = v.node_fp[node];
        HX_CHECK(ip >= 0 && ip <= v.ntab_p - 2 && it >= 0 && it <= v.ntab_t - 2 && node >= 0 && node < nnode, 1);
        w4[4 * s + 0] = (Real)((1.0 - fp) * (1.0 - ft) * ksc);
        w4[4 * s + 1] = (Real)((1.0 - fp) * ft * ksc);
        w4[4 * s + 2] = (Real)(fp * (1.0 - ft) * ksc);
        w4[4 * s + 3] = (Real)(fp * ft * ksc);
        noff[s] = (ip * v.ntab_t + it) * (v.nb * v.ng);
    }
    for (int s = tid; s < Sh::NSUB_PAD; s += blockDim.x) hPs[s] = (Real)((s < v.nsub) ? v.hP[s] : 0.0);
    for (int s = tid; s < kExpTab; s += blockDim.x) exp_tab[s] = exp2((double)s * (1.0 / kExpTab));
    // S15: the table is used when every node of the column lies below its end (same rule as the oracle)
    constexpr bool TAB = HX_FLUX_ALT != 0;      // variants 1 and 2 hold the table path
    bool use_ptab = false;
    if constexpr (TAB) {
        int nodes_in_table = 1;
        if (v.ptab)
            for (int s = tid; s < NN; s += blockDim.x)
                if (!(Tn[s] < v.ptab_Tmax)) nodes_in_table = 0;
        use_ptab = __syncthreads_and(nodes_in_table) != 0 && v.ptab != nullptr;
    }
    __syncthreads();

    const int base = sl * S;
    const bool base_odd = (base & 1) != 0;
    const int sl_top = (v.nsub - 1) / S, j_top = (v.nsub - 1) - sl_top * S;   // sub-lane / local index of the top sublayer
    constexpr bool ALT = HX_FLUX_ALT == 1;
    const bool exact = ALT && v.exact != 0;             // exact pure-absorption limit (S13): one pass, no coupling
    const bool direct = !exact && v.any_scat[0] && v.n_scat < 0;   // HELIOS_NSCAT_DIRECT: solve the coupled system (S12)
    const int n_sweeps = 1 + ((v.any_scat[0] && !direct && !exact) ? v.n_scat : 0);
    const double fs_scale = v.fs_scale[c];
    const double dtau_iso = fmax(v.dtau_iso, 1e-300);   // dtau = 0 (padding) always takes the isothermal form
    const size_t sT = (size_t)v.nb * v.ng, sP = sT * v.ntab_t;

    using R = AccRows<NACC, COMP>;
#pragma unroll
    for (int k = 0; k < R::ROWS; ++k) acc[32 * k] = 0.0;
    const bool want_spec = (v.spec_up_toa != nullptr) || (v.spec_dn_boa != nullptr);

    // This warp's run of units [u_lo, u_hi): unit u = (bin u / G, group u % G of 4 Gauss points), G groups per bin.
    // Batch plans: bins_per_warp whole bins.  unit_split plans: the block's units dealt evenly over its warps.
    const int G = (v.ng + kGroupG - 1) / kGroupG;
    int u_lo, u_hi;
    if (v.unit_split) {
        const int cb0 = (int)((long long)chunk * v.nb / v.n_chunks), cb1 = (int)((long long)(chunk + 1) * v.nb / v.n_chunks);
        const int U = (cb1 - cb0) * G;
        u_lo = cb0 * G + (int)((long long)warp * U / nwarps);
        u_hi = cb0 * G + (int)((long long)(warp + 1) * U / nwarps);
        if (lane == 0) { specbuf[6 * warp] = -1.0; specbuf[6 * warp + 3] = -1.0; }   // no spectrum shares yet
    } else {
        const int b_lo = chunk * v.bins_per_block + warp * v.bins_per_warp;
        const int b_hi = min(min(b_lo + v.bins_per_warp, (chunk + 1) * v.bins_per_block), v.nb);
        u_lo = b_lo * G;
        u_hi = max(b_hi, b_lo) * G;
    }
    const int bin_lo = u_lo / G, bin_hi = (u_hi > u_lo) ? (u_hi - 1) / G + 1 : bin_lo;
    // first / last Gauss point of the run in its first / last bin (fp64 form of the loop bounds below)
    const int g_first = (u_lo - bin_lo * G) * kGroupG, g_last = min((u_hi - (bin_hi - 1) * G) * kGroupG, v.ng);

    for (int bin = bin_lo; bin < bin_hi; ++bin) {
        const int grp_lo = (bin == bin_lo) ? u_lo - bin_lo * G : 0;       // this warp's groups of the bin
        const int grp_hi = (bin == bin_hi - 1) ? u_hi - bin * G : G;
        HX_CHECK(bin >= 0 && bin < v.nb && grp_lo >= 0 && grp_lo < grp_hi && grp_hi <= G, 2);
        // ---- (1) Planck (a2): lanes over nodes, node = lane + 32 j
        __syncwarp();
        if (TAB && use_ptab) {
            // tabulated Planck function (S15): linear in T between the nodes k * ptab_dT
            const double* __restrict__ row = v.ptab + (size_t)bin * v.ptab_n;
#pragma unroll
            for (int j = 0; j < NPL; ++j) {
                const int node = lane + 32 * j;
                if (node < NN) {
                    const double t = Tn[node] * v.ptab_inv_dT;
                    const int k = max((int)t, 0);
                    const double b0 = __ldg(row + k), b1 = __ldg(row + k + 1);
                    Bw[node] = (Real)(v.tpe * fma(t - (double)k, b1 - b0, b0));
                }
            }
        } else {
            if (bin == bin_lo) {
                double e_lo[NPL];
                planck_edges<NPL>(v.xedge[bin], Ti + lane, lane, NN, e_lo);
#pragma unroll
                for (int j = 0; j < NPL; ++j) Gw[32 * j] = e_lo[j];
            }
            const BinConst* bcp = v.bins + bin;
            const double pref = v.tpe * kPlanckPref / bcp->dnu;   // Bw = (2 pi / D) * bin-mean Planck
            double e_hi[NPL];
            planck_edges<NPL>(v.xedge[bin + 1], Ti + lane, lane, NN, e_hi);
#pragma unroll
            for (int j = 0; j < NPL; ++j) {
                const int node = lane + 32 * j;
                if (node < NN) {
                    const double T = Tn[node], T2 = T * T;
                    Bw[node] = (Real)(pref * T2 * T2 * planck_bin_integral(Gw[32 * j], e_hi[j]));
                }
                Gw[32 * j] = e_hi[j];
            }
        }
        __syncwarp();
        // per sublayer: mean and half difference of the end values (independent of the Gauss point)
#pragma unroll
        for (int j = 0; j < NSL; ++j) {
            const int s = lane + 32 * j;
            if (s < Sh::NSUB_PAD) {
                const Real lo = Bw[s], up = Bw[s + Sh::UP];
                Bmw[s] = Real(0.5) * (lo + up);
                Bhw[s] = Real(0.5) * (lo - up);
            }
        }

#ifdef HX_CHECKED
        __syncwarp();                                                 // B per node is dead now: poison the stage
        for (int i = lane; i < kGroupG * KLS; i += 32) kst[i] = Real(__longlong_as_double(-1ll));
#endif
        const BinConst bc = v.bins[bin];
        const double F_top = bc.fstar * fs_scale;                     // eq. 20
        const bool pure_scat = __shfl_sync(kFull, bc.pure_scat, 0) != 0;   // warp-uniform
        const double piB = v.piB_int[(size_t)c * v.nb + bin];        // eq. 21
        const BinConstF bcf(bc);
        const float dtau_iso_f = (float)dtau_iso;

        // The same bounds written in two ways: ptxas allocates the registers of the whole kernel differently for
        // them, and each arithmetic has its own winner (measured on config 4: fp64 101.1 vs 103.7 ms, fp32 53.7 vs 54.9 ms).
        const int g_begin = F32 ? grp_lo * kGroupG : ((bin == bin_lo) ? g_first : 0);
        const int g_end = F32 ? grp_hi * kGroupG : ((bin == bin_hi - 1) ? g_last : v.ng);
        for (int g0 = g_begin; g0 < g_end; g0 += kGroupG) {
            // ---- (2) kappa at every node for 4 Gauss points (a1)
            __syncwarp();
            stage_kappa<NN, KLS>(v, w4, noff, kst, bin, g0, lane, sT, sP);
            __syncwarp();
            // ---- (3) rays: RPW Gauss points at a time, one per group of LPR lanes
            const int ngg = min(kGroupG, v.ng - g0);
            for (int gg = 0; gg < ngg; gg += RPW) {
                const int gi = gg + rw;                         // this ray's row of the stage (rows beyond ngg repeat a valid g)
                const bool ray_on = gi < ngg;                   // else: an idle group of lanes, weight 0
                const int g = min(g0 + gi, v.ng - 1);
                HX_CHECK(gi >= 0 && gi < kGroupG && g >= 0 && base + S <= NN - 1 && gi * KLS + base + S < kGroupG * KLS, 3);
                Real a[S], b[S], su[S], sd[S];
                const Real* kp_ = kst + gi * KLS + base;
                bool coeffs_done = false;
                if constexpr (ALT) {
                    if (exact) {
                        ray_coefficients_exact<Real, S, ISO>(dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                        coeffs_done = true;
                    } else if (v.kscat) {                       // albedo per sublayer (S14)
                        const double kscb = v.kscat[bin], g0b = 1.0 - bc.xfac / v.D;
                        if (direct)
                            ray_coefficients_w0s<Real, S, ISO, true>(v.D, g0b, kscb, dtau_iso, v.omw_min, exp_tab, kp_, hPs + base,
                                                                     Bmw + base, Bhw + base, a, b, su, sd);
                        else
                            ray_coefficients_w0s<Real, S, ISO, false>(v.D, g0b, kscb, dtau_iso, v.omw_min, exp_tab, kp_, hPs + base,
                                                                      Bmw + base, Bhw + base, a, b, su, sd);
                        coeffs_done = true;
                    }
                }
                if constexpr (HX_FLUX_ALT == 2) {
                    if (v.tt_dlog > 0.0) {                       // tabulated transmission function (S16)
                        if (direct) {
                            if (pure_scat) ray_coefficients_tt<Real, S, ISO, true, true>(bc, v.tt_dlog, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                            else ray_coefficients_tt<Real, S, ISO, false, true>(bc, v.tt_dlog, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                        } else {
                            if (pure_scat) ray_coefficients_tt<Real, S, ISO, true, false>(bc, v.tt_dlog, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                            else ray_coefficients_tt<Real, S, ISO, false, false>(bc, v.tt_dlog, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                        }
                        coeffs_done = true;
                    }
                }
                if constexpr (F32 && S >= 4 && HX_FLUX_ALT == 0) {
                    // fp32 rays of an ordinary bin: coefficients in packed arithmetic (hx_ray.cuh); the sweeps from a cold
                    // start stay packed, the direct solve and the warm start take the same numbers as scalars.  Main
                    // variant only: with their extra paths the alt / tab kernels spill at 128 registers (measured:
                    // +26 % / +30 % time), so they keep the scalar forms.
                    if (!coeffs_done && !pure_scat) {
                        Packed2<S> C;
                        if (direct) ray_coefficients_f32_p2<S, ISO, true>(bcf, dtau_iso_f, kp_, hPs + base, Bmw + base, Bhw + base, C);
                        else ray_coefficients_f32_p2<S, ISO, false>(bcf, dtau_iso_f, kp_, hPs + base, Bmw + base, Bhw + base, C);
                        if (!direct && !v.warm_now) {
                            const double wgp = ray_on ? v.g_wts[g] : 0.0;
                            ray_sweeps_p2<S, LPR, ISO>(C, (Real)F_top, (Real)piB, n_sweeps, wgp * bc.dnu, wgp, sl, base_odd,
                                                       j_top, want_spec, acc);
                            continue;
                        }
#pragma unroll
                        for (int j = 0; j < S; ++j) {
                            constexpr int H = Packed2<S>::H;
                            a[j] = (Real)(j < H ? C.a[j < H ? j : 0].x : C.a[j >= H ? j - H : 0].y);
                            b[j] = (Real)(j < H ? C.b[j < H ? j : 0].x : C.b[j >= H ? j - H : 0].y);
                            su[j] = (Real)(j < H ? C.su[j < H ? j : 0].x : C.su[j >= H ? j - H : 0].y);
                            sd[j] = (Real)(j < H ? C.sd[j < H ? j : 0].x : C.sd[j >= H ? j - H : 0].y);
                        }
                        coeffs_done = true;
                    }
                }
                if (!coeffs_done && direct) {
                    if constexpr (F32) {
                        if (pure_scat) ray_coefficients_f32<S, ISO, true, true>(bcf, dtau_iso_f, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                        else ray_coefficients_f32<S, ISO, false, true>(bcf, dtau_iso_f, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                    } else {
                        if (pure_scat) ray_coefficients<S, ISO, true, true>(bc, exp_tab, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                        else ray_coefficients<S, ISO, false, true>(bc, exp_tab, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                    }
                    coeffs_done = true;
                }
                if (!coeffs_done) {
                    if constexpr (F32) {
                        if (pure_scat) ray_coefficients_f32<S, ISO, true>(bcf, dtau_iso_f, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                        else ray_coefficients_f32<S, ISO, false>(bcf, dtau_iso_f, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                    } else {
                        if (pure_scat) ray_coefficients<S, ISO, true>(bc, exp_tab, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                        else ray_coefficients<S, ISO, false>(bc, exp_tab, dtau_iso, kp_, hPs + base, Bmw + base, Bhw + base, a, b, su, sd);
                    }
                }
                const double wg = ray_on ? v.g_wts[g] : 0.0;
                Real* warm = nullptr;
                if (v.warm_now)
                    warm = reinterpret_cast<Real*>(v.fup_state) + (((size_t)c * v.nb + bin) * v.ng + g) * NN;
                if (direct)
                    ray_direct<Real, S, LPR, ISO>(a, b, su, sd, (Real)F_top, (Real)piB, wg * bc.dnu, wg, sl, base_odd,
                                                  j_top, want_spec, acc);
                else
                    ray_sweeps<Real, S, LPR, ISO>(a, b, su, sd, (Real)F_top, (Real)piB, n_sweeps, wg * bc.dnu, wg, sl,
                                                  base_odd, j_top, want_spec, acc, warm, ray_on);
            }
#ifdef HX_CHECKED
            __syncwarp();                                             // this group's kappa is dead: poison the stage
            for (int i = lane; i < kGroupG * KLS; i += 32) kst[i] = Real(__longlong_as_double(-1ll));
#endif
        }
        if (want_spec) {
            // the rays of a warp hold shares of the bin's sum over g: add them in ray order
            __syncwarp();
            double s_up = 0.0, s_dn = 0.0;
            if (lane == 0) {
#pragma unroll
                for (int r = 0; r < RPW; ++r) {
                    s_up += accw[32 * R::SPU + r * LPR + sl_top];
                    s_dn += accw[32 * R::SPD + r * LPR];
                }
                if (grp_lo == 0 && grp_hi == G) {      // the whole bin is this warp's
                    if (v.spec_up_toa) v.spec_up_toa[(size_t)c * v.nb + bin] = s_up;
                    if (v.spec_dn_boa) v.spec_dn_boa[(size_t)c * v.nb + bin] = s_dn;
                } else {     // this warp holds the sum over its share of the Gauss points only: combined below
                    HX_CHECK(v.unit_split && (bin == bin_lo || bin == bin_hi - 1), 4);
                    double* sb = specbuf + 6 * warp + ((bin == bin_lo) ? 0 : 3);
                    sb[0] = (double)bin;
                    sb[1] = s_up;
                    sb[2] = s_dn;
                }
            }
            __syncwarp();
            acc[32 * R::SPU] = 0.0;
            acc[32 * R::SPD] = 0.0;
        }
        if constexpr (COMP) {
            // end of the bin: add its sums to the running double-double sums (AccRows)
#pragma unroll
            for (int k = 0; k < R::NF; ++k) {
                double hi = acc[32 * (R::HI + k)], lo = acc[32 * (R::LO + k)];
                dd_add(hi, lo, acc[32 * k]);
                acc[32 * (R::HI + k)] = hi;
                acc[32 * (R::LO + k)] = lo;
                acc[32 * k] = 0.0;
            }
        }
    }

    // ---- a8: one partial per block = the warps' accumulator columns added in (warp, ray) order (deterministic).
    // Every (direction, interface) has exactly one owner (sub-lane, row) in each ray's lane group, so one thread
    // per (direction, interface) walks the warps' shared-memory columns in that order: no barrier per warp, and
    // the same association as adding the warps one after the other.
    __syncthreads();                      // every warp's accumulators are final
    {
        const unsigned char* wbase = smem_raw + Sm::BLOCK + Sm::W_ACC;
        for (int item = tid; item < 2 * (n + 1); item += blockDim.x) {
            const bool up = item <= n;
            const int j = up ? item : item - (n + 1);
            const int lev = j * v.lev_stride;
            int osl, row;                 // owner sub-lane and accumulator row of this level
            if (up) {                     // F_up at global level base + jl + 1 (up-sweep ownership); level 0: row UP0
                if (lev == 0) { osl = 0; row = R::UP0; }
                else { osl = (lev - 1) / S; const int jl = lev - 1 - osl * S; row = R::UP + (ISO ? jl : jl >> 1); }
            } else {                      // F_dn at global level base + jl; the top level: row DNT
                if (lev == NN - 1) { osl = LPR - 1; row = R::DNT; }
                else { osl = lev / S; const int jl = lev - osl * S; row = R::DN + (ISO ? jl : jl >> 1); }
            }
            HX_CHECK(lev < NN && osl >= 0 && osl < LPR && row >= 0 && row < R::NF, 8);
            double hi = 0.0, lo = 0.0;
            for (int w = 0; w < nwarps * RPW; ++w) {
                const double* col = reinterpret_cast<const double*>(wbase + (size_t)(w / RPW) * Sm::WARP) + (w % RPW) * LPR + osl;
                dd_add(hi, lo, col[32 * ((COMP ? R::HI : 0) + row)]);
                if (COMP) lo += col[32 * (R::LO + row)];
            }
            // partial[chunk][column][hi | lo][up | dn][n+1]
            double* out = v.partial + ((size_t)chunk * v.nc + c) * 4 * (n + 1);
            out[(up ? 0 : n + 1) + j] = hi;
            out[(up ? 2 : 3) * (n + 1) + j] = lo;
        }
    }
    if (want_spec && v.unit_split) {
        // per-bin spectra of the bins shared by several warps: add the warps' shares in warp order
        const int cb0 = (int)((long long)chunk * v.nb / v.n_chunks), cb1 = (int)((long long)(chunk + 1) * v.nb / v.n_chunks);
        for (int bin = cb0 + tid; bin < cb1; bin += blockDim.x) {
            double su = 0.0, sd = 0.0;
            bool shared = false;
            for (int e = 0; e < 2 * nwarps; ++e) {
                const double* sb = specbuf + 3 * e;
                if ((int)sb[0] == bin) { su += sb[1]; sd += sb[2]; shared = true; }
            }
            if (shared) {
                if (v.spec_up_toa) v.spec_up_toa[(size_t)c * v.nb + bin] = su;
                if (v.spec_dn_boa) v.spec_dn_boa[(size_t)c * v.nb + bin] = sd;
            }
        }
    }
#ifdef HX_CHECKED
    if (lane == 0) HX_CHECK(*reinterpret_cast<unsigned long long*>(wsm + Sm::WARP - 8) == 0x600DC0DE600DC0DEull, 5);
    if (tid == 0) HX_CHECK(*reinterpret_cast<unsigned long long*>(smem_raw + Sm::BLOCK - 8) == 0x600DC0DE600DC0DEull, 6);
    HX_CHECK(n * v.lev_stride <= NN - 1 && chunk < v.n_chunks && c < v.nc, 7);
#endif
}

template <int S, int LPR, bool ISO, typename Real>
int launch_one(const DevView& v, int respect_converged, cudaStream_t st)
{
    const size_t bytes = Smem<S, LPR, ISO, Real>::bytes(v.warps) + flux_spec_smem_bytes(v.warps, v.unit_split);
    dim3 grid(v.nc, v.n_chunks), block(32 * v.warps);
    k_flux<HX_FLUX_ALT, S, LPR, ISO, Real><<<grid, block, bytes, st>>>(v, respect_converged);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

template <int S, int LPR, bool ISO, typename Real>
int configure_one(size_t bytes)
{
    if (cudaFuncSetAttribute(k_flux<HX_FLUX_ALT, S, LPR, ISO, Real>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared) != cudaSuccess) return -1;
    return cudaFuncSetAttribute(k_flux<HX_FLUX_ALT, S, LPR, ISO, Real>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)bytes) == cudaSuccess ? 0 : -1;
}

// Shapes of this unit's LPR (flux_shape in helios_internal.h picks (LPR, S) from the number of sublayers):
// LPR = 8: S = 1 .. 13; LPR = 16: S = 7 .. 13; LPR = 32: S = 7 .. 16.
#ifdef HX_DEV_SHAPES   /* developer builds (build.py --dev): only the shapes of the BASELINE configs and the parity tests */
#if HX_FLUX_LPR == 8
#define HX_FOR_S(X) X(1) X(4) X(5) X(8) X(10) X(13)
#elif HX_FLUX_LPR == 16
#define HX_FOR_S(X) X(8) X(13)
#else
#define HX_FOR_S(X) X(13) X(16)
#endif
#else
#if HX_FLUX_LPR == 8
#define HX_FOR_S(X) X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13)
#elif HX_FLUX_LPR == 16
#define HX_FOR_S(X) X(7) X(8) X(9) X(10) X(11) X(12) X(13)
#else
#define HX_FOR_S(X) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16)
#endif
#endif

#if HX_FLUX_F32
using UnitReal = float;
#else
using UnitReal = double;
#endif
constexpr int kUnitLPR = HX_FLUX_LPR;

template <int S>
int configure_s(int iso, size_t bytes)
{
    return iso ? configure_one<S, kUnitLPR, true, UnitReal>(bytes) : configure_one<S, kUnitLPR, false, UnitReal>(bytes);
}
template <int S>
int launch_s(const DevView& v, int rc, cudaStream_t st)
{
    return v.iso ? launch_one<S, kUnitLPR, true, UnitReal>(v, rc, st) : launch_one<S, kUnitLPR, false, UnitReal>(v, rc, st);
}
template <int S>
size_t bytes_s(int warps, int iso)
{
    return iso ? Smem<S, kUnitLPR, true, UnitReal>::bytes(warps) : Smem<S, kUnitLPR, false, UnitReal>::bytes(warps);
}

}  // namespace unit_<variant>_<arithmetic>_<lanes per ray>
using namespace HX_UNIT_NAME(unit);

// entry points of this unit (declared in helios_internal.h, routed by helios_flux_dispatch.cu)
int HX_UNIT_NAME(flux_configure)(int S, int iso, size_t smem_bytes)
{
    switch (S) {
#define X(s) case s: return configure_s<s>(iso, smem_bytes);
        HX_FOR_S(X)
#undef X
    }
    return -1;
}

int HX_UNIT_NAME(launch_flux)(const DevView& v, int respect_converged, cudaStream_t st)
{
    switch (v.S) {
#define X(s) case s: return launch_s<s>(v, respect_converged, st);
        HX_FOR_S(X)
#undef X
    }
    return -1;
}

#if HX_FLUX_ALT == 0   /* the shared-memory size of a shape does not depend on the variant */
size_t HX_UNIT_NAME(flux_smem)(int S, int warps, int iso)
{
    switch (S) {
#define X(s) case s: return bytes_s<s>(warps, iso);
        HX_FOR_S(X)
#undef X
    }
    return 0;
}
#endif

}  // namespace hx
