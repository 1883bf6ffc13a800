// helios_internal.h -- structures shared by the C-ABI host code and the CUDA kernels.
// Product code: shares nothing with oracle/.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/helios.h"

namespace hx {

// Physical constants, cgs (CODATA 2018 exact SI values).
constexpr double kH = 6.62607015e-27;    // erg s
constexpr double kC = 2.99792458e10;     // cm s^-1
constexpr double kKB = 1.380649e-16;     // erg K^-1
constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kC2 = kH * kC / kKB;    // second radiation constant, cm K
// Planck prefactor 2 k^4/(h^3 c^2): B_bin = kPlanckPref T^4 * Int/dnu
constexpr double kPlanckPref = 2.0 * (kKB * kKB) * (kKB * kKB) / ((kH * kH) * kH * (kC * kC));
// sigma_SB = 2 pi^5 k^4 / (15 h^3 c^2)
constexpr double kSigmaSB = kPlanckPref * (kPi * kPi) * (kPi * kPi) * kPi / 15.0;

constexpr int kGroupG = 4;        // Gauss points staged together (4 fp64 = one 32-byte sector)
constexpr int kMaxS = 16;         // sublayers per lane
constexpr int kMaxSNarrow = 13;   // ... when a ray takes 8 or 16 lanes (several rays per warp)

// Lay-out of a ray of nsub sublayers: LPR lanes x S sublayers per lane (hx_ray.cuh).  The narrowest ray that
// holds the column in <= 13 sublayers per lane: more rays per warp share every shuffle of the scan, the scan
// has fewer rounds and less of the lane grid is padding (100 layers: 16 x 13 = 208 slots for 200 sublayers).
struct FluxShape { int lpr, S; };
inline FluxShape flux_shape(int nsub)
{
    for (int lpr = 8; lpr <= 16; lpr *= 2)
        if (nsub <= lpr * kMaxSNarrow) return {lpr, (nsub + lpr - 1) / lpr};
    return {32, (nsub + 31) / 32};
}

// Warps per block of the ray kernel = the register budget of a shape (__launch_bounds__): fp64 168 registers
// (12 warps) up to S = 7, 255 (8 warps) above; fp32 ray arithmetic 96 (20 warps) / 128 (16 warps).
// (Measured on config 4: two blocks of 4 warps per SM instead of one of 8: 375.9 vs 365.1 ms; fp32 with 8 / 10 / 12 /
// 16 warps, i.e. 212 / 168 / 166 / 128 registers: 258.6 / 251.3 / 224.9 / 204.4 ms -- occupancy beats registers there.)
template <int S, bool F32> struct FluxWarps {
    static constexpr int value = F32 ? (S <= 7 ? 20 : 16) : (S <= 7 ? 12 : 8);
};
inline int flux_warps_max(int S, int precision)
{
    return precision == HELIOS_PREC_FP32 ? (S <= 7 ? 20 : 16) : (S <= 7 ? 12 : 8);
}

// Per-bin constants of eq. 8, 12-14: everything that depends on (w0, g0, D) only.
struct BinConst {
    double nlam_tab; // -256 lambda log2(e), lambda = D sqrt((1-w0 g0)(1-w0))  (eq. 8; exp2 with a 2^(j/256) table)
    double zp2;     // zeta_+^2                                           (eq. 13)
    double zm2;     // zeta_-^2
    double zpzm;    // zeta_+ zeta_-
    double zp, zm;  // zeta_+, zeta_-
    double lam;     // lambda
    double r;       // sqrt((1-w0)/(1-w0 g0)) = zeta_+ - zeta_-;  xi = -r*T
    double kp;      // eps/(1 - w0 g0)                                    (eq. 15, reading G2)
    double xfac;    // D (1-g0)                                           (eq. 14)
    double dnu;     // bin width, cm^-1
    double fstar;   // TOA downward flux per unit wavenumber (eq. 20), before the column scale
    int32_t pure_scat;  // 1 - w0 < one_minus_w0_min
    int32_t pad_;
};

// The same constants in fp32 registers (fp32 ray arithmetic).
struct BinConstF {
    float nlam2, lam, zp, zm, zpzm, r, kp, xfac;
    __host__ __device__ explicit BinConstF(const BinConst& b)
        : nlam2((float)(b.nlam_tab * (1.0 / 256.0))), lam((float)b.lam), zp((float)b.zp), zm((float)b.zm),
          zpzm((float)b.zpzm), r((float)b.r), kp((float)b.kp), xfac((float)b.xfac) {}
};

// Device-side view of one context: dimensions + pointers into the workspace.
struct DevView {
    // dimensions
    int nc, n, nb, ng, ntab_p, ntab_t;
    int nsub;        // sublayers: 2n (non-isothermal) or n
    int nnode;       // opacity/Planck nodes: 2n+1 levels, or n layer centres
    int iso;         // isothermal_layers
    int lev_stride;  // flux level of interface j = j*lev_stride
    int S;           // sublayers per lane
    int lpr;         // lanes per ray (8, 16, 32)
    int n_scat;
    int precision;   // HELIOS_PREC_FP64 / HELIOS_PREC_FP32
    int bins_per_block, bins_per_warp, n_chunks, warps;
    int unit_split;  // small-batch plan: block q takes the bins [q nb / n_chunks, (q+1) nb / n_chunks) and its warps share
                     // the block's (bin, group of 4 Gauss points) units in contiguous, equally long runs; else a warp owns
                     // bins_per_warp whole bins of the block's bins_per_block
    int exact;       // exact_absorption: eq. 3/4/6 instead of the two-stream coefficients
    const double* kscat;   // [nb] scattering opacity per bin (helios_set_scattering, reading S14) or NULL
    const double* ptab;    // [nb][ptab_n] bin-mean Planck function at T_k = k * ptab_dT (reading S15) or NULL
    int ptab_n;
    double ptab_dT, ptab_inv_dT, ptab_Tmax;
    double tt_dlog;  // trans_table_dlog10k (reading S16) or 0
    double omw_min;  // one_minus_w0_min
    double D, tpe /* 2 pi / D */, dtau_iso, dT_frac_max, T_floor, flux_floor;
    // setup arrays
    const double* ktab;        // [ntab_p][ntab_t][nb][ng]  (caller's)
    const float* ktab32;       // fp32 copy of the table (workspace; fp32 precision only)
    const double* tab_axis;    // [2] tab_t[0], (ntab_t-1)/(tab_t[last]-tab_t[0])
    const double* g_wts;       // [ng]
    const double* xedge;       // [nb+1]  c2 * bin_edges
    const double* edges;       // [nb+1]  bin_edges (copy)
    const BinConst* bins;      // [nb]
    const double* hP;          // [nsub]  (P_lo - P_up)/(2 gravity)
    const int32_t* node_ip;    // [nnode] table P cell
    const double* node_fp;     // [nnode] table P weight
    const double* w_iface;     // [n+1]   T_interface = T[a] + w (T[b]-T[a])
    const double* p_layer;     // [n]
    const double* p_ratio;     // [n]     P_i / (P_int,i - P_int,i+1)
    const int32_t* any_scat;   // [1]
    // per-column state
    double* T;                 // [nc][n]
    const double* fs_scale;    // [nc]
    const double* kscale;      // [nc]
    const double* t_intern;    // [nc]
    const double* piB_int;     // [nc][nb]  pi * B_bin(T_intern)
    double* step_factor;       // [nc][n]
    int32_t* sign_hist;        // [nc][n]
    double* dT_last;           // [nc][n]
    int32_t* iters;            // [nc]
    int32_t* converged;        // [nc]
    int32_t* n_running;        // [1] columns not yet converged
    int32_t* nonfinite;        // [1]
    int32_t* check_fail;       // [1] HX_CHECKED builds: code of a failed check of the ray kernel (0 = none)
    int32_t* col_nonfinite;    // [nc] this column produced a non-finite flux / step (cleared per call)
    double* col_max_dT;        // [nc] max_i |dT_i| of the column's last RE iteration
    double* col_max_rel;       // [nc] max_i |dF_i| / (sigma T_i^4) of it (eq. 29)
    // outputs of the ray kernel and of the reduction
    void* fup_state;           // warm start: [nc][nb][ng][32 S + 1] F_up per level (double / float), else NULL
    int warm_now;              // this launch starts from fup_state and updates it
    double* partial;           // [n_chunks][nc][hi | lo][up | dn][n+1] double-double partial sums
    double* F_up;              // [nc][n+1]
    double* F_dn;              // [nc][n+1]
    double* spec_up_toa;       // [nc][nb] or NULL (caller's)
    double* spec_dn_boa;       // [nc][nb] or NULL (caller's)
};

// launchers (defined in the .cu files); each returns the number of kernels launched (>= 0) or -1
// after recording a CUDA error.
int launch_setup_levels(const helios_params& p, const double* p_layer, const double* p_interface,
                        const double* tab_log10p, const double* tab_t, double* hP, int32_t* node_ip,
                        double* node_fp, double* w_iface, double* p_ratio, double* tab_axis_out,
                        cudaStream_t st);
int launch_setup_bins(const helios_params& p, const double* bin_edges, const double* w0,
                      const double* g0, double* xedge, double* edges_copy, BinConst* bins,
                      int32_t* any_scat, cudaStream_t st);
int launch_set_fstar(int nb, const double* f_star, BinConst* bins, cudaStream_t st);
int launch_planck_intern(const DevView& v, double* piB_int, cudaStream_t st);
int launch_build_planck_table(const DevView& v, double* tab, cudaStream_t st);
int launch_set_kscat(int nb, const double* src, double* dst, int32_t* any_scat, cudaStream_t st);
int launch_reset_re(const DevView& v, cudaStream_t st);
int launch_fill(double* p, size_t count, double value, cudaStream_t st);
int launch_count_running(const DevView& v, cudaStream_t st);
int launch_clear_nonfinite(const DevView& v, cudaStream_t st);
int launch_flux(const DevView& v, int respect_converged, cudaStream_t st);
int launch_reduce(const DevView& v, int do_re, int respect_converged, double tol_dT, double tol_flux,
                  cudaStream_t st);
// helios_flux_dispatch.cu: routes to the unit (variant, arithmetic, lanes per ray) that holds the kernel
size_t flux_smem_bytes(int lpr, int S, int warps, int iso, int precision);
size_t flux_spec_smem_bytes(int warps, int unit_split);
int launch_convert_table(const double* src, float* dst, size_t count, cudaStream_t st);
int flux_configure(int lpr, int S, int iso, int precision, size_t smem_bytes);   // cudaFuncSetAttribute (all variants)
double measure_fma_peak(int precision, int distinct_operands, cudaStream_t st);

}  // namespace hx
