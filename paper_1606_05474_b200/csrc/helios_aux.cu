// helios_aux.cu -- the small kernels around the ray kernel: set-up of per-level / per-bin constants,
// pi*B(T_intern), the chunk reduction with the radiative-equilibrium temperature step (a8-a9), and
// the FMA-rate microbenchmark used as the ALU roofline denominator.
// Product code (CUDA path, sm_100a); shares nothing with oracle/.
#include "helios_internal.h"
#include "hx_math.cuh"

namespace hx {

namespace {

// ---------------------------------------------------------------------------------------------
// set-up
// ---------------------------------------------------------------------------------------------
__global__ void k_setup_levels(helios_params p, const double* __restrict__ p_layer,
                               const double* __restrict__ p_interface,
                               const double* __restrict__ tab_log10p,
                               const double* __restrict__ tab_t, double* __restrict__ hP,
                               int32_t* __restrict__ node_ip, double* __restrict__ node_fp,
                               double* __restrict__ w_iface, double* __restrict__ p_ratio,
                               double* __restrict__ tab_axis)
{
    const int n = p.n_layers;
    const int iso = p.isothermal_layers;
    const int nnode = iso ? n : 2 * n + 1, nsub = iso ? n : 2 * n;
    const int t0 = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    const double lp0 = tab_log10p[0];
    const double dlp = (tab_log10p[p.ntab_p - 1] - lp0) / (double)(p.ntab_p - 1);
    auto node_p = [&](int v) -> double {
        if (iso) return p_layer[v];
        return (v & 1) ? p_layer[v >> 1] : p_interface[v >> 1];
    };
    for (int v = t0; v < nnode; v += stride) {                 // table P cell and weight
        double tp = (log10(node_p(v)) - lp0) / dlp;
        tp = fmin(fmax(tp, 0.0), (double)(p.ntab_p - 1));
        const int ip = min((int)tp, p.ntab_p - 2);
        node_ip[v] = ip;
        node_fp[v] = tp - (double)ip;
    }
    for (int s = t0; s < nsub; s += stride) {                   // eq. 19 without kappa
        const double dP = iso ? (p_interface[s] - p_interface[s + 1]) : (node_p(s) - node_p(s + 1));
        hP[s] = dP / p.gravity * 0.5;
    }
    for (int j = t0; j <= n; j += stride) {                     // interface T weights
        double w = 0.0;
        if (n > 1) {
            int a = j - 1, b = j;
            if (j == 0) { a = 0; b = 1; }
            if (j == n) { a = n - 2; b = n - 1; }
            const double la = log(p_layer[a]), lb = log(p_layer[b]), lj = log(p_interface[j]);
            w = (lj - la) / (lb - la);
        }
        w_iface[j] = w;
    }
    for (int i = t0; i < n; i += stride) p_ratio[i] = p_layer[i] / (p_interface[i] - p_interface[i + 1]);
    if (t0 == 0) {
        tab_axis[0] = tab_t[0];
        tab_axis[1] = (double)(p.ntab_t - 1) / (tab_t[p.ntab_t - 1] - tab_t[0]);
    }
}

__global__ void k_setup_bins(helios_params p, const double* __restrict__ bin_edges,
                             const double* __restrict__ w0, const double* __restrict__ g0,
                             double* __restrict__ xedge, double* __restrict__ edges_copy,
                             BinConst* __restrict__ bins, int32_t* __restrict__ any_scat)
{
    const int t0 = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    for (int e = t0; e <= p.n_bins; e += stride) {
        xedge[e] = kC2 * bin_edges[e];
        edges_copy[e] = bin_edges[e];
    }
    for (int l = t0; l < p.n_bins; l += stride) {
        const double w = w0[l], g = g0[l], D = p.D;
        BinConst bc;
        const double omw = 1.0 - w, omwg = 1.0 - w * g;
        const double r = sqrt(omw / omwg);                       // eq. 13
        const double zp = 0.5 * (1.0 + r), zm = 0.5 * (1.0 - r);
        const double lam = D * sqrt(omwg * omw);                 // eq. 8
        bc.nlam_tab = -lam * 1.44269504088896340735992468100 * 256.0;
        bc.zp2 = zp * zp;
        bc.zm2 = zm * zm;
        bc.zpzm = zp * zm;
        bc.zp = zp;
        bc.zm = zm;
        bc.lam = lam;
        bc.r = r;
        bc.kp = (1.0 / D) / omwg;                                // reading G2
        bc.xfac = D * (1.0 - g);                                 // eq. 14
        bc.dnu = bin_edges[l + 1] - bin_edges[l];
        bc.fstar = bins[l].fstar;                                // kept (set by k_set_fstar)
        bc.pure_scat = (omw < p.one_minus_w0_min) ? 1 : 0;
        bc.pad_ = 0;
        bins[l] = bc;
        if (w > 0.0) atomicOr(any_scat, 1);
    }
}

__global__ void k_set_fstar(int nb, const double* __restrict__ f_star, BinConst* __restrict__ bins)
{
    for (int l = blockIdx.x * blockDim.x + threadIdx.x; l < nb; l += gridDim.x * blockDim.x)
        bins[l].fstar = f_star[l];
}

// scattering opacity per bin (helios_set_scattering): copy into the workspace; any value > 0 switches the
// scattering sweeps on (w0 of setup is not used from then on, so the flag is recomputed, not or-ed)
__global__ void k_set_kscat(int nb, const double* __restrict__ src, double* __restrict__ dst, int32_t* __restrict__ any_scat)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        int any = 0;
        for (int l = 0; l < nb; ++l) {
            dst[l] = src[l];
            if (src[l] > 0.0) any = 1;
        }
        *any_scat = any;
    }
}

// -H(x) below x = kPlanckSwitch, G(x) above (see hx_math.cuh)
__device__ inline double planck_edge_scalar(double x)
{
    return (x < kPlanckSwitch) ? -planck_lower(x) : planck_upper(x);
}

// pi * bin-mean Planck function at T_intern (eq. 21): [nc][nb]
__global__ void k_planck_intern(DevView v, double* __restrict__ piB)
{
    const size_t total = (size_t)v.nc * v.nb;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total;
         i += (size_t)gridDim.x * blockDim.x) {
        const int c = (int)(i / v.nb), l = (int)(i % v.nb);
        const double T = v.t_intern[c];
        double out = 0.0;
        if (T > 0.0) {
            const double e_lo = planck_edge_scalar(v.xedge[l] / T);
            const double e_hi = planck_edge_scalar(v.xedge[l + 1] / T);
            const double T2 = T * T;
            out = kPi * kPlanckPref * T2 * T2 * planck_bin_integral(e_lo, e_hi) / v.bins[l].dnu;
        }
        piB[i] = out;
    }
}

// Planck table of reading S15: tab[l][k] = bin-mean Planck function of bin l at T_k = k * ptab_dT
__global__ void k_build_planck_table(DevView v, double* __restrict__ tab)
{
    const size_t total = (size_t)v.nb * v.ptab_n;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total;
         i += (size_t)gridDim.x * blockDim.x) {
        const int l = (int)(i / v.ptab_n), k = (int)(i % v.ptab_n);
        const double T = (double)k * v.ptab_dT;
        double out = 0.0;
        if (T > 0.0) {
            const double e_lo = planck_edge_scalar(v.xedge[l] / T);
            const double e_hi = planck_edge_scalar(v.xedge[l + 1] / T);
            const double T2 = T * T;
            out = kPlanckPref * T2 * T2 * planck_bin_integral(e_lo, e_hi) / v.bins[l].dnu;
        }
        tab[i] = out;
    }
}

__global__ void k_reset_re(DevView v)
{
    const size_t total = (size_t)v.nc * v.n;
    const size_t t0 = blockIdx.x * (size_t)blockDim.x + threadIdx.x, stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = t0; i < total; i += stride) {
        v.step_factor[i] = 1.0;
        v.sign_hist[i] = 0;
        v.dT_last[i] = 0.0;
    }
    for (size_t c = t0; c < (size_t)v.nc; c += stride) {
        v.iters[c] = 0;
        v.converged[c] = 0;
        v.col_nonfinite[c] = 0;
        v.col_max_dT[c] = 0.0;
        v.col_max_rel[c] = 0.0;
    }
    if (t0 == 0) {
        v.n_running[0] = v.nc;
        v.nonfinite[0] = 0;
    }
}

__global__ void k_clear_nonfinite(DevView v)
{
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < v.nc; c += gridDim.x * blockDim.x) v.col_nonfinite[c] = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) v.nonfinite[0] = 0;
}

__global__ void k_count_running(DevView v)
{
    __shared__ int cnt;
    if (threadIdx.x == 0) cnt = 0;
    __syncthreads();
    int mine = 0;
    for (int c = threadIdx.x; c < v.nc; c += blockDim.x) mine += (v.converged[c] || v.col_nonfinite[c]) ? 0 : 1;
    atomicAdd(&cnt, mine);
    __syncthreads();
    if (threadIdx.x == 0) v.n_running[0] = cnt;
}

__global__ void k_convert_table(const double* __restrict__ src, float* __restrict__ dst, size_t count)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < count;
         i += (size_t)gridDim.x * blockDim.x)
        dst[i] = (float)src[i];
}

__global__ void k_fill(double* __restrict__ p, size_t count, double value)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < count;
         i += (size_t)gridDim.x * blockDim.x)
        p[i] = value;
}

// ---------------------------------------------------------------------------------------------
// a8 (chunk reduction) + a9 (radiative-equilibrium step): one block per column
// ---------------------------------------------------------------------------------------------

// sign history packing documented in include/helios.h
__device__ __forceinline__ int32_t hist_push(int32_t h, double dT)
{
    const int32_t code = dT > 0.0 ? 1 : (dT < 0.0 ? 2 : 0);
    int32_t cnt = (h >> 12) & 0xF;
    cnt = min(cnt + 1, 6);
    return (cnt << 12) | ((h << 2) & 0xFFC) | code;
}

// PAPER.md:309-311 (reading S7): x0.67 if the last six steps strictly alternate, x1.1 if all six
// have the same non-zero sign.
__device__ __forceinline__ double hist_factor(int32_t h)
{
    if (((h >> 12) & 0xF) < 6) return 1.0;
    const int32_t codes = h & 0xFFF;
    if (codes == 0x555 || codes == 0xAAA) return 1.1;          // 010101010101b / 101010101010b
    if (codes == 0x666 || codes == 0x999) return 0.67;         // 1,2,1,2,1,2 / 2,1,2,1,2,1
    return 1.0;
}

__global__ void __launch_bounds__(1024)
k_reduce(DevView v, int do_re, int respect_converged, double tol_dT, double tol_flux, int slices)
{
    extern __shared__ double sh[];          // [n+1] net flux, [64] max scratch, [slices][4][n+1] partial sums
    const int c = blockIdx.x, n = v.n, tid = threadIdx.x;
    if (respect_converged && (v.converged[c] || v.col_nonfinite[c])) return;   // a flagged column is left untouched
    double* fnet = sh;
    double* smax = sh + (n + 1);
    double* part = smax + 64;
    const int nl = n + 1;
    bool bad = false;                       // this thread met a non-finite flux or step
    // partial[chunk][column][hi | lo][up | dn][n+1]: double-double partial sums of the ray kernel's blocks,
    // added here with compensation as well (dd_add), always in the same order: bit-reproducible
    if (slices > 1) {
        // many chunks (single columns): slice s adds chunks s, s+slices, ... in order; the slices are
        // then added in order -- a fixed association
        const int per = blockDim.x / slices;                      // threads per slice (>= 1)
        const int s = tid / per, t = tid - s * per;
        if (s < slices) {
            for (int j = t; j < nl; j += per) {
                double up = 0.0, dn = 0.0, ul = 0.0, dl = 0.0;
                for (int q = s; q < v.n_chunks; q += slices) {
                    const double* pp = v.partial + ((size_t)q * v.nc + c) * 4 * nl;
                    dd_add(up, ul, pp[j]);
                    dd_add(dn, dl, pp[nl + j]);
                    ul += pp[2 * nl + j];
                    dl += pp[3 * nl + j];
                }
                part[(4 * s) * nl + j] = up;
                part[(4 * s + 1) * nl + j] = dn;
                part[(4 * s + 2) * nl + j] = ul;
                part[(4 * s + 3) * nl + j] = dl;
            }
        }
        __syncthreads();
    }
    for (int j = tid; j <= n; j += blockDim.x) {
        double up = 0.0, dn = 0.0, ul = 0.0, dl = 0.0;
        if (slices > 1) {
            for (int s = 0; s < slices; ++s) {
                dd_add(up, ul, part[(4 * s) * nl + j]);
                dd_add(dn, dl, part[(4 * s + 1) * nl + j]);
                ul += part[(4 * s + 2) * nl + j];
                dl += part[(4 * s + 3) * nl + j];
            }
        } else {
            for (int q = 0; q < v.n_chunks; ++q) {               // fixed order: deterministic
                const double* pp = v.partial + ((size_t)q * v.nc + c) * 4 * nl;
                dd_add(up, ul, pp[j]);
                dd_add(dn, dl, pp[nl + j]);
                ul += pp[2 * nl + j];
                dl += pp[3 * nl + j];
            }
        }
        up += ul;
        dn += dl;
        v.F_up[(size_t)c * (n + 1) + j] = up;
        v.F_dn[(size_t)c * (n + 1) + j] = dn;
        fnet[j] = up - dn;                                       // eq. 23: net flux
        if (!isfinite(up) || !isfinite(dn)) bad = true;
    }
    if (!do_re) {
        if (bad) { v.nonfinite[0] = 1; v.col_nonfinite[c] = 1; }
        return;
    }
    __syncthreads();

    double* Tc = v.T + (size_t)c * n;
    double my_dT = 0.0, my_rel = 0.0;
    for (int i = tid; i < n; i += blockDim.x) {
        double dF = fnet[i + 1] - fnet[i];                      // eq. 23
        const double T = Tc[i];
        // dead zone (S11): a layer that meets eq. 29 locally is in equilibrium, dF := 0
        if (fabs(dF) < v.flux_floor * (kSigmaSB * T * T * T * T)) dF = 0.0;
        const double a = v.step_factor[(size_t)c * n + i];
        double dT = 0.0;
        if (dF != 0.0) {                                          // eq. 24-28 collapsed (S6), sign G3
            const double mag = pow(fabs(dF), 0.1);
            dT = -a * 1.0e5 * v.p_ratio[i] * (dF > 0.0 ? mag : -mag) / (kSigmaSB * T * T * T);
        }
        const double lim = v.dT_frac_max * T;                    // limiter (S7)
        if (!isfinite(dT) || !isfinite(T)) bad = true;           // before the limiter: fmin/fmax would swallow a NaN
        else dT = fmin(fmax(dT, -lim), lim);
        v.dT_last[(size_t)c * n + i] = dT;
        my_dT = fmax(my_dT, fabs(dT));
        my_rel = fmax(my_rel, fabs(dF) / (kSigmaSB * T * T * T * T));   // eq. 29
    }
    // block max
    for (int o = 16; o > 0; o >>= 1) {
        my_dT = fmax(my_dT, __shfl_xor_sync(0xffffffffu, my_dT, o));
        my_rel = fmax(my_rel, __shfl_xor_sync(0xffffffffu, my_rel, o));
    }
    if ((tid & 31) == 0) { smax[tid >> 5] = my_dT; smax[32 + (tid >> 5)] = my_rel; }
    if (__syncthreads_or(bad)) {            // the column is flagged and left as it is; the others carry on
        if (tid == 0) { v.nonfinite[0] = 1; v.col_nonfinite[c] = 1; v.iters[c] += 1; atomicSub(v.n_running, 1); }
        return;
    }
    double max_dT = 0.0, max_rel = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
        max_dT = fmax(max_dT, smax[w]);
        max_rel = fmax(max_rel, smax[32 + w]);
    }
    const bool conv = (tol_dT > 0.0 && max_dT < tol_dT) || (tol_flux > 0.0 && max_rel < tol_flux);
    if (tid == 0) {
        v.iters[c] += 1;
        v.col_max_dT[c] = max_dT;
        v.col_max_rel[c] = max_rel;
        if (conv) {
            v.converged[c] = 1;
            atomicSub(v.n_running, 1);
        }
    }
    if (conv) return;
    for (int i = tid; i < n; i += blockDim.x) {
        const size_t k = (size_t)c * n + i;
        const double dT = v.dT_last[k];
        Tc[i] = fmax(Tc[i] + dT, v.T_floor);
        const int32_t h = hist_push(v.sign_hist[k], dT);
        v.sign_hist[k] = h;
        v.step_factor[k] *= hist_factor(h);
    }
}

// ---------------------------------------------------------------------------------------------
// FMA issue-rate microbenchmark (roofline denominator): 8 independent register chains per thread
// ---------------------------------------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(256) k_fma_peak(R* out, int iters, R seed)
{
    R x0 = seed + (R)threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5,
      x6 = x0 + 6, x7 = x0 + 7;
    const R m = (R)0.999, b = (R)0.001;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fma(x0, m, b); x1 = fma(x1, m, b); x2 = fma(x2, m, b); x3 = fma(x3, m, b);
            x4 = fma(x4, m, b); x5 = fma(x5, m, b); x6 = fma(x6, m, b); x7 = fma(x7, m, b);
        }
    }
    const R s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == (R)-1) out[0] = s;     // never true; keeps the chains alive
}

// The same with three distinct register operands per FMA (y_i, z_i differ per chain): an FP64 FMA then
// reads six 32-bit registers, and the register file, not the FP64 pipe, sets the issue rate.
template <typename R>
__global__ void __launch_bounds__(256) k_fma3_peak(R* out, int iters, R seed)
{
    R x[8], y[8], z[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        x[i] = seed + (R)(threadIdx.x + i);
        y[i] = (R)0.999 + (R)1e-6 * (R)(threadIdx.x + i);
        z[i] = (R)1e-3 * (R)(i + 1) + (R)1e-7 * (R)threadIdx.x;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = fma(x[i], y[i], z[i]);
        }
    }
    R s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == (R)-1) out[0] = s;
}

inline int grid_for(size_t count, int block = 256)
{
    size_t g = (count + block - 1) / block;
    if (g < 1) g = 1;
    if (g > 148 * 16) g = 148 * 16;
    return (int)g;
}

inline int ok() { return cudaPeekAtLastError() == cudaSuccess ? 1 : -1; }

}  // namespace

int launch_setup_levels(const helios_params& p, const double* p_layer, const double* p_interface,
                        const double* tab_log10p, const double* tab_t, double* hP, int32_t* node_ip,
                        double* node_fp, double* w_iface, double* p_ratio, double* tab_axis_out,
                        cudaStream_t st)
{
    k_setup_levels<<<grid_for(2 * (size_t)p.n_layers + 1), 256, 0, st>>>(
        p, p_layer, p_interface, tab_log10p, tab_t, hP, node_ip, node_fp, w_iface, p_ratio, tab_axis_out);
    return ok();
}

int launch_setup_bins(const helios_params& p, const double* bin_edges, const double* w0,
                      const double* g0, double* xedge, double* edges_copy, BinConst* bins,
                      int32_t* any_scat, cudaStream_t st)
{
    k_setup_bins<<<grid_for((size_t)p.n_bins + 1), 256, 0, st>>>(p, bin_edges, w0, g0, xedge, edges_copy,
                                                                 bins, any_scat);
    return ok();
}

int launch_set_fstar(int nb, const double* f_star, BinConst* bins, cudaStream_t st)
{
    k_set_fstar<<<grid_for((size_t)nb), 256, 0, st>>>(nb, f_star, bins);
    return ok();
}

int launch_build_planck_table(const DevView& v, double* tab, cudaStream_t st)
{
    k_build_planck_table<<<grid_for((size_t)v.nb * v.ptab_n), 256, 0, st>>>(v, tab);
    return ok();
}

int launch_set_kscat(int nb, const double* src, double* dst, int32_t* any_scat, cudaStream_t st)
{
    k_set_kscat<<<1, 32, 0, st>>>(nb, src, dst, any_scat);
    return ok();
}

int launch_planck_intern(const DevView& v, double* piB_int, cudaStream_t st)
{
    k_planck_intern<<<grid_for((size_t)v.nc * v.nb), 256, 0, st>>>(v, piB_int);
    return ok();
}

int launch_reset_re(const DevView& v, cudaStream_t st)
{
    k_reset_re<<<grid_for((size_t)v.nc * v.n), 256, 0, st>>>(v);
    return ok();
}

int launch_fill(double* p, size_t count, double value, cudaStream_t st)
{
    k_fill<<<grid_for(count), 256, 0, st>>>(p, count, value);
    return ok();
}

int launch_convert_table(const double* src, float* dst, size_t count, cudaStream_t st)
{
    k_convert_table<<<grid_for(count), 256, 0, st>>>(src, dst, count);
    return ok();
}

int launch_clear_nonfinite(const DevView& v, cudaStream_t st)
{
    k_clear_nonfinite<<<grid_for((size_t)v.nc), 256, 0, st>>>(v);
    return ok();
}

int launch_count_running(const DevView& v, cudaStream_t st)
{
    k_count_running<<<1, 256, 0, st>>>(v);
    return ok();
}

int launch_reduce(const DevView& v, int do_re, int respect_converged, double tol_dT, double tol_flux,
                  cudaStream_t st)
{
    int threads = v.n + 1 > 128 ? 256 : 128, slices = 1;
    if (v.n_chunks >= 16) {                 // single-column shapes: spread the chunk sum over the block
        slices = 8;                         // ... within the default 48 KB of dynamic shared memory
        while (slices > 1 && sizeof(double) * (((size_t)v.n + 1) + 64 + (size_t)slices * 4 * (v.n + 1)) > 40 * 1024) slices >>= 1;
        if (slices > 1) threads = 1024;
    }
    const size_t sh = sizeof(double) * (((size_t)v.n + 1) + 64 + (slices > 1 ? (size_t)slices * 4 * (v.n + 1) : 0));
    k_reduce<<<v.nc, threads, sh, st>>>(v, do_re, respect_converged, tol_dT, tol_flux, slices);
    return ok();
}

double measure_fma_peak(int precision, int distinct_operands, cudaStream_t st)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return (double)HELIOS_E_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return (double)HELIOS_E_CUDA;
    void* out = nullptr;
    if (cudaMalloc(&out, 64) != cudaSuccess) return (double)HELIOS_E_CUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256, iters = precision == HELIOS_PREC_FP32 ? 8192 : 4096;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        if (distinct_operands) {
            if (precision == HELIOS_PREC_FP32) k_fma3_peak<float><<<blocks, threads, 0, st>>>((float*)out, iters, 1.0f);
            else k_fma3_peak<double><<<blocks, threads, 0, st>>>((double*)out, iters, 1.0);
        } else {
            if (precision == HELIOS_PREC_FP32) k_fma_peak<float><<<blocks, threads, 0, st>>>((float*)out, iters, 1.0f);
            else k_fma_peak<double><<<blocks, threads, 0, st>>>((double*)out, iters, 1.0);
        }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = (double)HELIOS_E_CUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fmas = (double)blocks * threads * (double)iters * 64.0;
        if (rep > 0 && ms > 0.f) best = fmax(best, fmas / (ms * 1e-3));
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return best;
}

}  // namespace hx
