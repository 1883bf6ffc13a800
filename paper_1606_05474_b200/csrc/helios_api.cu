// helios_api.cu -- the C-ABI of include/helios.h: argument checks, workspace lay-out, launch
// sequencing.  No arithmetic of the method lives here; every step runs in the kernels of
// helios_flux.cu / helios_aux.cu.  Product code; shares nothing with oracle/.
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "helios_internal.h"

using namespace hx;

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

// Launch plan + workspace offsets; a pure function of the parameters so that
// helios_workspace_bytes and helios_setup agree.
struct Plan {
    int nsub, nnode, lpr, S, warps, n_chunks, bins_per_block, bins_per_warp, unit_split;
    size_t smem;
    // offsets (bytes)
    size_t o_tab_axis, o_gwts, o_xedge, o_edges, o_bins, o_hP, o_node_ip, o_node_fp, o_w_iface,
        o_p_layer, o_p_ratio, o_flags, o_T, o_fs_scale, o_kscale, o_t_intern, o_piB, o_step,
        o_hist, o_dT, o_iters, o_conv, o_colnf, o_colmax, o_colrel, o_partial, o_Fup, o_Fdn, o_stage, o_ktab32, o_kscat, o_ptab, o_fup, total;
    int ptab_n;
};

bool params_ok(const helios_params* p, const char** why)
{
    *why = "";
    if (!p) { *why = "params is NULL"; return false; }
    if (p->n_cols < 1 || p->n_layers < 1 || p->n_bins < 1 || p->n_g < 1) { *why = "sizes must be >= 1"; return false; }
    if (p->ntab_p < 2 || p->ntab_t < 2) { *why = "k-table needs at least 2 nodes per axis"; return false; }
    if (p->precision != HELIOS_PREC_FP64 && p->precision != HELIOS_PREC_FP32) { *why = "precision must be HELIOS_PREC_FP64 or HELIOS_PREC_FP32"; return false; }
    if (p->n_scat < 0 && p->n_scat != HELIOS_NSCAT_DIRECT) { *why = "n_scat < 0 (other than HELIOS_NSCAT_DIRECT)"; return false; }
    if (p->n_scat == HELIOS_NSCAT_DIRECT && p->warm_start) { *why = "warm_start has no meaning with the direct solve"; return false; }
    if (p->warm_start != 0 && p->warm_start != 1) { *why = "warm_start must be 0 or 1"; return false; }
    if (p->isothermal_layers != 0 && p->isothermal_layers != 1) { *why = "isothermal_layers must be 0 or 1"; return false; }
    const long nsub = p->isothermal_layers ? p->n_layers : 2L * p->n_layers;
    if (nsub > HELIOS_MAX_SUBLAYERS) { *why = "too many sublayers (HELIOS_MAX_SUBLAYERS)"; return false; }
    if (!(p->D > 0.0) || !(p->gravity > 0.0)) { *why = "D and gravity must be > 0"; return false; }
    if (!(p->dtau_iso >= 0.0) || !(p->one_minus_w0_min >= 0.0)) { *why = "thresholds must be >= 0"; return false; }
    if (!(p->flux_floor >= 0.0)) { *why = "flux_floor must be >= 0"; return false; }
    if (!(p->planck_table_dT >= 0.0)) { *why = "planck_table_dT must be >= 0"; return false; }
    if (p->planck_table_dT > 0.0 && (!(p->planck_table_Tmax > p->planck_table_dT) ||
                                     p->planck_table_Tmax / p->planck_table_dT > 1.0e6)) {
        *why = "planck_table_Tmax must exceed planck_table_dT (at most 1e6 nodes)"; return false;
    }
    if (!(p->trans_table_dlog10k >= 0.0) || (p->trans_table_dlog10k > 0.0 && p->trans_table_dlog10k < 1.0e-6)) {
        *why = "trans_table_dlog10k must be 0 or >= 1e-6"; return false;
    }
    if (p->trans_table_dlog10k > 0.0 && p->exact_absorption) { *why = "trans_table_dlog10k has no meaning in the exact pure-absorption limit"; return false; }
    if (p->exact_absorption != 0 && p->exact_absorption != 1) { *why = "exact_absorption must be 0 or 1"; return false; }
    if (p->exact_absorption && p->warm_start) { *why = "warm_start has no meaning in the pure-absorption limit"; return false; }
    if (!(p->dT_frac_max > 0.0) || !(p->T_floor > 0.0)) { *why = "dT_frac_max and T_floor must be > 0"; return false; }
    if (p->warm_start) {   // per-ray upward fluxes persist in the workspace: only for batches that fit
        const long ns = p->isothermal_layers ? p->n_layers : 2L * p->n_layers;
        const FluxShape sh = flux_shape((int)ns);
        const double state_bytes = (double)p->n_cols * p->n_bins * p->n_g * ((double)sh.lpr * sh.S + 1) * 8.0;
        if (state_bytes > 16.0 * 1073741824.0) { *why = "warm_start: per-ray flux state exceeds 16 GiB (DESIGN.md S4)"; return false; }
    }
    const double tab_elems = (double)p->ntab_p * p->ntab_t * (double)p->n_bins * p->n_g;
    if (tab_elems >= 2147483648.0) { *why = "k-table has >= 2^31 elements"; return false; }
    return true;
}

Plan make_plan(const helios_params& p)
{
    Plan L{};
    L.nsub = p.isothermal_layers ? p.n_layers : 2 * p.n_layers;
    L.nnode = p.isothermal_layers ? p.n_layers : 2 * p.n_layers + 1;
    const FluxShape shape = flux_shape(L.nsub);
    L.lpr = shape.lpr;
    L.S = shape.S;
    // warps per block: bounded by the registers of the shape and by shared memory (227 KB per block on sm_100a)
    const size_t smem_max = 227 * 1024;
    int wmax = flux_warps_max(L.S, p.precision);
    while (wmax > 1 && flux_smem_bytes(L.lpr, L.S, wmax, p.isothermal_layers, p.precision) > smem_max) --wmax;
    // small batches: split the bins over enough blocks to fill the 148 SMs, but never more than one
    // wave of them (a block of this kernel owns most of an SM's shared memory)
    long chunks = 148 / p.n_cols;
    if (chunks < 1) {
        // batches: blocks are dispatched column-fastest within a bin chunk (grid = (columns, chunks)), so
        // the blocks in flight read the same slice of the k-table; chunks of <= 32 MiB keep that slice
        // resident in L2 (HBM then sees the table once per evaluation) as long as a warp keeps >= 8 bins
        const double tab_bytes = (double)p.ntab_p * p.ntab_t * (double)p.n_bins * p.n_g * (p.precision == HELIOS_PREC_FP32 ? 4.0 : 8.0);
        chunks = (long)(tab_bytes / (32.0 * 1048576.0) + 0.999);
        const long most = p.n_bins / (8L * wmax);
        if (chunks > most) chunks = most;
        if (chunks > 65535) chunks = 65535;
        if (chunks >= 1) {
            // a block takes as long as its fullest warp: among chunk counts up to twice the minimum pick the one
            // whose bins split most evenly over the warps (1000 bins, 8 warps: 5 chunks of 8 x 25, not 4 of 7 x 32 + 26)
            long best = chunks, best_slots = -1;
            for (long q = chunks; q <= 2 * chunks && q <= most; ++q) {
                const long bpb = (p.n_bins + q - 1) / q, bpw = (bpb + wmax - 1) / wmax;
                const long slots = bpw * wmax * ((p.n_bins + bpb - 1) / bpb);      // warp-bins paid for
                if (best_slots < 0 || slots < best_slots) { best = q; best_slots = slots; }
            }
            chunks = best;
        }
    }
    const bool small_batch = chunks >= 1 && p.n_cols <= 148;
    if (chunks < 1) chunks = 1;
    if (chunks > p.n_bins) chunks = p.n_bins;
    L.unit_split = 0;
    if (small_batch) {
        // small batches (single columns) are latency-bound: one wave of blocks, block q takes the bins
        // [q nb / n_chunks, (q+1) nb / n_chunks) (sizes differ by at most one), and the block's (bin, group of 4 Gauss
        // points) units, bin-major, are dealt to its warps in contiguous, equally long runs -- a warp may start in
        // the middle of a bin and end in the middle of another (config 1: 148 blocks of 2-3 bins = 10-15 units over
        // 8 warps, at most 2 units = 4 ray pairs per warp)
        const int groups = (p.n_g + kGroupG - 1) / kGroupG;
        L.unit_split = 1;
        L.n_chunks = (int)chunks;
        L.bins_per_block = (int)((p.n_bins + chunks - 1) / chunks);      // the largest block
        const long units = (long)L.bins_per_block * groups;
        L.warps = (int)(units < wmax ? units : wmax);
        L.bins_per_warp = L.bins_per_block;                               // a warp's run lies within the block's bins
        while (L.warps > 1 && flux_smem_bytes(L.lpr, L.S, L.warps, p.isothermal_layers, p.precision) +
                                  flux_spec_smem_bytes(L.warps, L.unit_split) > smem_max) --L.warps;
    } else {
        L.bins_per_block = (int)((p.n_bins + chunks - 1) / chunks);
        L.n_chunks = (p.n_bins + L.bins_per_block - 1) / L.bins_per_block;
        int w = L.bins_per_block < wmax ? L.bins_per_block : wmax;
        L.bins_per_warp = (L.bins_per_block + w - 1) / w;
        L.warps = (L.bins_per_block + L.bins_per_warp - 1) / L.bins_per_warp;
    }
    L.smem = flux_smem_bytes(L.lpr, L.S, L.warps, p.isothermal_layers, p.precision) +
             flux_spec_smem_bytes(L.warps, L.unit_split);

    const size_t nc = p.n_cols, n = p.n_layers, nb = p.n_bins, ng = p.n_g;
    size_t o = 0;
    auto take = [&](size_t bytes) { const size_t at = o; o = align_up(o + bytes); return at; };
    L.o_tab_axis = take(2 * 8);
    L.o_gwts = take(ng * 8);
    L.o_xedge = take((nb + 1) * 8);
    L.o_edges = take((nb + 1) * 8);
    L.o_bins = take(nb * sizeof(BinConst));
    L.o_hP = take((size_t)L.nsub * 8);
    L.o_node_ip = take((size_t)L.nnode * 4);
    L.o_node_fp = take((size_t)L.nnode * 8);
    L.o_w_iface = take((n + 1) * 8);
    L.o_p_layer = take(n * 8);
    L.o_p_ratio = take(n * 8);
    L.o_flags = take(4 * 4);              // any_scat, n_running, nonfinite, spare
    L.o_T = take(nc * n * 8);
    L.o_fs_scale = take(nc * 8);
    L.o_kscale = take(nc * 8);
    L.o_t_intern = take(nc * 8);
    L.o_piB = take(nc * nb * 8);
    L.o_step = take(nc * n * 8);
    L.o_hist = take(nc * n * 4);
    L.o_dT = take(nc * n * 8);
    L.o_iters = take(nc * 4);
    L.o_conv = take(nc * 4);
    L.o_colnf = take(nc * 4);
    L.o_colmax = take(nc * 8);
    L.o_colrel = take(nc * 8);
    L.o_partial = take((size_t)L.n_chunks * nc * 4 * (n + 1) * 8);   // double-double pairs
    L.o_Fup = take(nc * (n + 1) * 8);
    L.o_Fdn = take(nc * (n + 1) * 8);
    L.o_stage = take((nb > nc ? nb : nc) * 8);   // staging for host f_star
    L.o_ktab32 = take(p.precision == HELIOS_PREC_FP32 ? (size_t)p.ntab_p * p.ntab_t * nb * ng * 4 : 0);
    L.o_kscat = take(nb * 8);
    L.ptab_n = p.planck_table_dT > 0.0 ? (int)(p.planck_table_Tmax / p.planck_table_dT) + 2 : 0;
    L.o_ptab = take(nb * (size_t)L.ptab_n * 8);
    L.o_fup = take(p.warm_start ? nc * nb * ng * (size_t)(L.lpr * L.S + 1) * (p.precision == HELIOS_PREC_FP32 ? 4 : 8) : 0);
    L.total = o;
    return L;
}

}  // namespace

// Scratch of helios_fluxes_static (include/helios.h): the ray kernel's per-block partial sums for callers that
// must not allocate.  In host code this name is only a stand-in for the symbol, not a device address: the address
// comes from cudaGetSymbolAddress (static_scratch_of_current_device below), once per device.
static __device__ __align__(256) unsigned char g_static_scratch[HELIOS_STATIC_SCRATCH_BYTES];

struct helios_ctx {
    int device;            // the device that was current at helios_setup
    void* static_scratch;  // device address of g_static_scratch on it (NULL if the look-up failed)
    helios_params p;
    Plan plan;
    DevView v;
    cudaStream_t st;
    char* ws;
    bool columns_set;
    int64_t launches;
    int32_t* h_flags;      // pinned: [0] n_running, [1] nonfinite
    // CUDA-graph replay of the RE loop: batches of g_batch (k_flux, k_reduce) pairs captured on an
    // internal stream that is ordered after/before the caller's stream with events
    cudaStream_t gst;
    cudaEvent_t g_in, g_out;
    cudaGraphExec_t gexec;
    double g_tol_dT, g_tol_flux;
    int g_batch;
    bool timing;
    std::vector<cudaEvent_t> ev;   // pairs (start, stop) of the ray-kernel launches since the last read
    size_t ev_used;
    char err[256];
};

namespace {

int fail(helios_ctx* c, int code, const char* msg)
{
    if (c) snprintf(c->err, sizeof c->err, "%s", msg);
    return code;
}

int fail_cuda(helios_ctx* c, const char* where)
{
    const cudaError_t e = cudaGetLastError();
    if (c) snprintf(c->err, sizeof c->err, "%s: %s", where, cudaGetErrorString(e));
    return HELIOS_E_CUDA;
}

#define HX_LAUNCH(ctx, call)                                  \
    do {                                                      \
        const int k_ = (call);                                \
        if (k_ < 0) return fail_cuda((ctx), #call);           \
        (ctx)->launches += k_;                                \
    } while (0)

#define HX_CUDA(ctx, call)                                    \
    do {                                                      \
        if ((call) != cudaSuccess) return fail_cuda((ctx), #call); \
    } while (0)

constexpr size_t kMaxEventPairs = 4096;

// launches the ray kernel, bracketed by events when timing is on
int flux_launch(helios_ctx* ctx, int respect_converged)
{
    const bool rec = ctx->timing && ctx->ev_used < kMaxEventPairs;
    if (rec) {
        if (ctx->ev.size() < 2 * (ctx->ev_used + 1)) {
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return -1;
            ctx->ev.push_back(a);
            ctx->ev.push_back(b);
        }
        if (cudaEventRecord(ctx->ev[2 * ctx->ev_used], ctx->st) != cudaSuccess) return -1;
    }
    const int k = launch_flux(ctx->v, respect_converged, ctx->st);
    if (rec) {
        if (cudaEventRecord(ctx->ev[2 * ctx->ev_used + 1], ctx->st) != cudaSuccess) return -1;
        ctx->ev_used++;
    }
    return k;
}

template <typename T>
T* at(helios_ctx* c, size_t off) { return reinterpret_cast<T*>(c->ws + off); }

char g_noctx_err[128] = "";

int copy_columns(helios_ctx* ctx, const double* T, const double* f_star, const double* f_star_scale,
                 const double* t_intern, const double* kscale, cudaMemcpyKind kind)
{
    const helios_params& p = ctx->p;
    const Plan& L = ctx->plan;
    if (!T || !f_star || !t_intern) return fail(ctx, HELIOS_E_BADARG, "T, f_star and t_intern must not be NULL");
    const size_t nc = p.n_cols, n = p.n_layers, nb = p.n_bins;
    HX_CUDA(ctx, cudaMemcpyAsync(ctx->ws + L.o_T, T, nc * n * 8, kind, ctx->st));
    HX_CUDA(ctx, cudaMemcpyAsync(ctx->ws + L.o_t_intern, t_intern, nc * 8, kind, ctx->st));
    if (f_star_scale) HX_CUDA(ctx, cudaMemcpyAsync(ctx->ws + L.o_fs_scale, f_star_scale, nc * 8, kind, ctx->st));
    else HX_LAUNCH(ctx, launch_fill(at<double>(ctx, L.o_fs_scale), nc, 1.0, ctx->st));
    if (kscale) HX_CUDA(ctx, cudaMemcpyAsync(ctx->ws + L.o_kscale, kscale, nc * 8, kind, ctx->st));
    else HX_LAUNCH(ctx, launch_fill(at<double>(ctx, L.o_kscale), nc, 1.0, ctx->st));
    HX_CUDA(ctx, cudaMemcpyAsync(ctx->ws + L.o_stage, f_star, nb * 8, kind, ctx->st));
    HX_LAUNCH(ctx, launch_set_fstar(p.n_bins, at<double>(ctx, L.o_stage), at<BinConst>(ctx, L.o_bins), ctx->st));
    HX_LAUNCH(ctx, launch_planck_intern(ctx->v, at<double>(ctx, L.o_piB), ctx->st));
    HX_LAUNCH(ctx, launch_reset_re(ctx->v, ctx->st));
    if (p.warm_start)   // the first evaluation of a warm-started run is a cold one: F_up = 0
        HX_CUDA(ctx, cudaMemsetAsync(ctx->ws + L.o_fup, 0, L.total - L.o_fup, ctx->st));
    ctx->columns_set = true;
    return HELIOS_OK;
}

int check_flags(helios_ctx* ctx, cudaStream_t st)
{
    HX_CUDA(ctx, cudaMemcpyAsync(ctx->h_flags, ctx->ws + ctx->plan.o_flags + 4, 12, cudaMemcpyDeviceToHost, st));
    HX_CUDA(ctx, cudaStreamSynchronize(st));
    if (ctx->h_flags[2]) {      // only HX_CHECKED builds ever set it
        snprintf(ctx->err, sizeof ctx->err, "checked build: ray-kernel check %d failed", ctx->h_flags[2]);
        return HELIOS_E_CUDA;
    }
    return HELIOS_OK;
}
int check_flags(helios_ctx* ctx) { return check_flags(ctx, ctx->st); }

// (Re)builds the graph of `batch` RE iterations for these tolerances.
int ensure_graph(helios_ctx* ctx, int batch, double tol_dT, double tol_flux)
{
    if (ctx->gexec && ctx->g_batch == batch && ctx->g_tol_dT == tol_dT && ctx->g_tol_flux == tol_flux) return HELIOS_OK;
    if (ctx->gexec) { cudaGraphExecDestroy(ctx->gexec); ctx->gexec = nullptr; }
    cudaGraph_t graph = nullptr;
    HX_CUDA(ctx, cudaStreamBeginCapture(ctx->gst, cudaStreamCaptureModeThreadLocal));
    bool ok = true;
    for (int k = 0; k < batch && ok; ++k) {
        ok = launch_flux(ctx->v, 1, ctx->gst) >= 0;
        ok = ok && launch_reduce(ctx->v, 1, 1, tol_dT, tol_flux, ctx->gst) >= 0;
    }
    const cudaError_t e = cudaStreamEndCapture(ctx->gst, &graph);
    if (!ok || e != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        return fail_cuda(ctx, "graph capture of the RE loop");
    }
    const cudaError_t e2 = cudaGraphInstantiate(&ctx->gexec, graph, 0);
    cudaGraphDestroy(graph);
    if (e2 != cudaSuccess) { ctx->gexec = nullptr; return fail_cuda(ctx, "cudaGraphInstantiate"); }
    ctx->g_batch = batch;
    ctx->g_tol_dT = tol_dT;
    ctx->g_tol_flux = tol_flux;
    return HELIOS_OK;
}

// Device address of g_static_scratch on the current device, looked up once per device (NULL on failure).
void* static_scratch_of_current_device(int* device_out)
{
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static void* ptr[kMaxDev] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); *device_out = -1; return nullptr; }
    *device_out = dev;
    if (dev < 0 || dev >= kMaxDev) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        ptr[dev] = p;
    }
    return ptr[dev];
}

}  // namespace

extern "C" {

size_t helios_workspace_bytes(const helios_params* params)
{
    const char* why;
    if (!params_ok(params, &why)) return 0;
    return make_plan(*params).total;
}

int helios_setup(helios_ctx** out, const helios_params* params,
                 const double* p_layer, const double* p_interface, const double* bin_edges,
                 const double* g_pts, const double* g_wts, const double* ktab,
                 const double* tab_log10p, const double* tab_t,
                 const double* w0, const double* g0,
                 void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (out) *out = nullptr;
    const char* why;
    if (!out) { snprintf(g_noctx_err, sizeof g_noctx_err, "out is NULL"); return HELIOS_E_BADARG; }
    if (!params_ok(params, &why)) { snprintf(g_noctx_err, sizeof g_noctx_err, "%s", why); return HELIOS_E_BADARG; }
    if (!p_layer || !p_interface || !bin_edges || !g_pts || !g_wts || !ktab || !tab_log10p || !tab_t || !w0 || !g0) {
        snprintf(g_noctx_err, sizeof g_noctx_err, "a setup array is NULL");
        return HELIOS_E_BADARG;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        snprintf(g_noctx_err, sizeof g_noctx_err, "no CUDA device (there is no CPU fallback)");
        return HELIOS_E_CUDA;
    }
    const Plan L = make_plan(*params);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) % kAlign) != 0 || workspace_bytes < L.total) {
        snprintf(g_noctx_err, sizeof g_noctx_err, "workspace NULL, misaligned or too small (%zu needed)", L.total);
        return HELIOS_E_WORKSPACE;
    }
    helios_ctx* ctx = new (std::nothrow) helios_ctx();
    if (!ctx) { snprintf(g_noctx_err, sizeof g_noctx_err, "out of host memory"); return HELIOS_E_BADARG; }
    ctx->p = *params;
    ctx->plan = L;
    ctx->st = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->ws = static_cast<char*>(workspace);
    ctx->columns_set = false;
    ctx->launches = 0;
    ctx->err[0] = 0;
    ctx->h_flags = nullptr;
    ctx->timing = false;
    ctx->ev_used = 0;
    ctx->gst = nullptr;
    ctx->g_in = ctx->g_out = nullptr;
    ctx->gexec = nullptr;
    ctx->g_batch = 0;
    ctx->g_tol_dT = ctx->g_tol_flux = 0.0;
    ctx->static_scratch = static_scratch_of_current_device(&ctx->device);   // helios_fluxes_static only
    if (cudaStreamCreateWithFlags(&ctx->gst, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->g_in, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->g_out, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        ctx->gst = nullptr;           // graphs are an optimisation: fall back to plain launches
    }
    auto bail = [&](int code) { const int r = code; snprintf(g_noctx_err, sizeof g_noctx_err, "%s", ctx->err);
                                if (ctx->h_flags) cudaFreeHost(ctx->h_flags);
                                if (ctx->g_in) cudaEventDestroy(ctx->g_in);
                                if (ctx->g_out) cudaEventDestroy(ctx->g_out);
                                if (ctx->gst) cudaStreamDestroy(ctx->gst);
                                delete ctx; return r; };
    if (cudaHostAlloc(reinterpret_cast<void**>(&ctx->h_flags), 64, cudaHostAllocDefault) != cudaSuccess)
        return bail(fail_cuda(ctx, "cudaHostAlloc"));
    if (L.smem > 227 * 1024) return bail(fail(ctx, HELIOS_E_BADARG, "ray kernel needs more than 227 KB of shared memory"));
    if (L.smem == 0 || flux_configure(L.lpr, L.S, params->isothermal_layers, params->precision, L.smem) != 0)
        return bail(fail_cuda(ctx, "cudaFuncSetAttribute"));

    const helios_params& p = ctx->p;
    DevView& v = ctx->v;
    memset(&v, 0, sizeof v);
    v.nc = p.n_cols; v.n = p.n_layers; v.nb = p.n_bins; v.ng = p.n_g; v.ntab_p = p.ntab_p; v.ntab_t = p.ntab_t;
    v.nsub = L.nsub; v.nnode = L.nnode; v.iso = p.isothermal_layers; v.lev_stride = p.isothermal_layers ? 1 : 2;
    v.S = L.S; v.lpr = L.lpr; v.n_scat = p.n_scat; v.precision = p.precision;
    v.bins_per_block = L.bins_per_block; v.bins_per_warp = L.bins_per_warp; v.n_chunks = L.n_chunks; v.warps = L.warps; v.unit_split = L.unit_split;
    v.exact = p.exact_absorption;
    v.kscat = nullptr;
    v.ptab = L.ptab_n ? at<double>(ctx, L.o_ptab) : nullptr;
    v.ptab_n = L.ptab_n;
    v.ptab_dT = p.planck_table_dT; v.ptab_inv_dT = L.ptab_n ? 1.0 / p.planck_table_dT : 0.0; v.ptab_Tmax = p.planck_table_Tmax;
    v.tt_dlog = p.trans_table_dlog10k;
    v.omw_min = p.one_minus_w0_min;
    v.D = p.D; v.tpe = p.exact_absorption ? kPi : 2.0 * kPi / p.D;   // eq. 3/4 carry pi B, eq. 11/15 2 pi eps B
    v.dtau_iso = p.dtau_iso; v.dT_frac_max = p.dT_frac_max; v.T_floor = p.T_floor; v.flux_floor = p.flux_floor;
    v.ktab = ktab;
    v.ktab32 = p.precision == HELIOS_PREC_FP32 ? at<float>(ctx, L.o_ktab32) : nullptr;
    v.fup_state = p.warm_start ? (void*)(ctx->ws + L.o_fup) : nullptr;
    v.warm_now = 0;
    v.tab_axis = at<double>(ctx, L.o_tab_axis);
    v.g_wts = at<double>(ctx, L.o_gwts);
    v.xedge = at<double>(ctx, L.o_xedge);
    v.edges = at<double>(ctx, L.o_edges);
    v.bins = at<BinConst>(ctx, L.o_bins);
    v.hP = at<double>(ctx, L.o_hP);
    v.node_ip = at<int32_t>(ctx, L.o_node_ip);
    v.node_fp = at<double>(ctx, L.o_node_fp);
    v.w_iface = at<double>(ctx, L.o_w_iface);
    v.p_layer = at<double>(ctx, L.o_p_layer);
    v.p_ratio = at<double>(ctx, L.o_p_ratio);
    v.any_scat = at<int32_t>(ctx, L.o_flags);
    v.n_running = at<int32_t>(ctx, L.o_flags) + 1;
    v.nonfinite = at<int32_t>(ctx, L.o_flags) + 2;
    v.check_fail = at<int32_t>(ctx, L.o_flags) + 3;
    v.T = at<double>(ctx, L.o_T);
    v.fs_scale = at<double>(ctx, L.o_fs_scale);
    v.kscale = at<double>(ctx, L.o_kscale);
    v.t_intern = at<double>(ctx, L.o_t_intern);
    v.piB_int = at<double>(ctx, L.o_piB);
    v.step_factor = at<double>(ctx, L.o_step);
    v.sign_hist = at<int32_t>(ctx, L.o_hist);
    v.dT_last = at<double>(ctx, L.o_dT);
    v.iters = at<int32_t>(ctx, L.o_iters);
    v.converged = at<int32_t>(ctx, L.o_conv);
    v.col_nonfinite = at<int32_t>(ctx, L.o_colnf);
    v.col_max_dT = at<double>(ctx, L.o_colmax);
    v.col_max_rel = at<double>(ctx, L.o_colrel);
    v.partial = at<double>(ctx, L.o_partial);
    v.F_up = at<double>(ctx, L.o_Fup);
    v.F_dn = at<double>(ctx, L.o_Fdn);

    // zero the small-array region (flags, bins.fstar) and copy what is used verbatim
    if (cudaMemsetAsync(ctx->ws, 0, L.o_T, ctx->st) != cudaSuccess) return bail(fail_cuda(ctx, "cudaMemsetAsync"));
    if (cudaMemcpyAsync(ctx->ws + L.o_gwts, g_wts, (size_t)p.n_g * 8, cudaMemcpyDeviceToDevice, ctx->st) != cudaSuccess ||
        cudaMemcpyAsync(ctx->ws + L.o_p_layer, p_layer, (size_t)p.n_layers * 8, cudaMemcpyDeviceToDevice, ctx->st) != cudaSuccess)
        return bail(fail_cuda(ctx, "cudaMemcpyAsync(setup)"));
    int k = launch_setup_levels(p, p_layer, p_interface, tab_log10p, tab_t, at<double>(ctx, L.o_hP),
                                at<int32_t>(ctx, L.o_node_ip), at<double>(ctx, L.o_node_fp),
                                at<double>(ctx, L.o_w_iface), at<double>(ctx, L.o_p_ratio),
                                at<double>(ctx, L.o_tab_axis), ctx->st);
    if (k < 0) return bail(fail_cuda(ctx, "k_setup_levels"));
    ctx->launches += k;
    k = launch_setup_bins(p, bin_edges, w0, g0, at<double>(ctx, L.o_xedge), at<double>(ctx, L.o_edges),
                          at<BinConst>(ctx, L.o_bins), at<int32_t>(ctx, L.o_flags), ctx->st);
    if (k < 0) return bail(fail_cuda(ctx, "k_setup_bins"));
    ctx->launches += k;
    if (L.ptab_n) {
        k = launch_build_planck_table(ctx->v, at<double>(ctx, L.o_ptab), ctx->st);
        if (k < 0) return bail(fail_cuda(ctx, "k_build_planck_table"));
        ctx->launches += k;
    }
    if (p.precision == HELIOS_PREC_FP32) {
        k = launch_convert_table(ktab, at<float>(ctx, L.o_ktab32), (size_t)p.ntab_p * p.ntab_t * p.n_bins * p.n_g, ctx->st);
        if (k < 0) return bail(fail_cuda(ctx, "k_convert_table"));
        ctx->launches += k;
    }
    (void)g_pts;   // the nodes enter only through the table's g axis; the weights do the quadrature
    *out = ctx;
    return HELIOS_OK;
}

int helios_set_columns(helios_ctx* ctx, const double* T, const double* f_star,
                       const double* f_star_scale, const double* t_intern, const double* kscale)
{
    if (!ctx) return HELIOS_E_BADARG;
    return copy_columns(ctx, T, f_star, f_star_scale, t_intern, kscale, cudaMemcpyDeviceToDevice);
}

int helios_set_columns_host(helios_ctx* ctx, const double* T, const double* f_star,
                            const double* f_star_scale, const double* t_intern, const double* kscale)
{
    if (!ctx) return HELIOS_E_BADARG;
    const int r = copy_columns(ctx, T, f_star, f_star_scale, t_intern, kscale, cudaMemcpyHostToDevice);
    if (r != HELIOS_OK) return r;
    HX_CUDA(ctx, cudaStreamSynchronize(ctx->st));
    return HELIOS_OK;
}

int helios_set_scattering(helios_ctx* ctx, const double* kappa_scat)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!kappa_scat) return fail(ctx, HELIOS_E_BADARG, "kappa_scat is NULL");
    if (ctx->p.exact_absorption) return fail(ctx, HELIOS_E_BADARG, "no scattering in the exact pure-absorption limit");
    if (ctx->p.trans_table_dlog10k > 0.0) return fail(ctx, HELIOS_E_BADARG, "the tabulated transmission function is per bin: not with a scattering opacity per sublayer");
    double* dst = at<double>(ctx, ctx->plan.o_kscat);
    HX_LAUNCH(ctx, launch_set_kscat(ctx->p.n_bins, kappa_scat, dst, at<int32_t>(ctx, ctx->plan.o_flags), ctx->st));
    ctx->v.kscat = dst;
    if (ctx->gexec) { cudaGraphExecDestroy(ctx->gexec); ctx->gexec = nullptr; }   // the captured launches hold the old view
    return HELIOS_OK;
}

int helios_set_temperatures(helios_ctx* ctx, const double* T)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!T) return fail(ctx, HELIOS_E_BADARG, "T is NULL");
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    HX_CUDA(ctx, cudaMemcpyAsync(ctx->ws + ctx->plan.o_T, T, (size_t)ctx->p.n_cols * ctx->p.n_layers * 8,
                                 cudaMemcpyDeviceToDevice, ctx->st));
    return HELIOS_OK;
}

int helios_fluxes(helios_ctx* ctx, double* F_up, double* F_dn, double* spec_up_toa, double* spec_dn_boa)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const size_t fb = (size_t)ctx->p.n_cols * (ctx->p.n_layers + 1) * 8;
    ctx->v.spec_up_toa = spec_up_toa;
    ctx->v.spec_dn_boa = spec_dn_boa;
    ctx->v.warm_now = 0;                       // one-shot evaluations are cold
    HX_LAUNCH(ctx, launch_clear_nonfinite(ctx->v, ctx->st));
    const int k_flux_launched = flux_launch(ctx, 0);
    ctx->v.spec_up_toa = nullptr;
    ctx->v.spec_dn_boa = nullptr;
    HX_LAUNCH(ctx, k_flux_launched);
    HX_LAUNCH(ctx, launch_reduce(ctx->v, 0, 0, 0.0, 0.0, ctx->st));
    if (F_up) HX_CUDA(ctx, cudaMemcpyAsync(F_up, ctx->v.F_up, fb, cudaMemcpyDeviceToDevice, ctx->st));
    if (F_dn) HX_CUDA(ctx, cudaMemcpyAsync(F_dn, ctx->v.F_dn, fb, cudaMemcpyDeviceToDevice, ctx->st));
    return HELIOS_OK;
}

int helios_fluxes_static(helios_ctx* ctx, double* F_up, double* F_dn)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const size_t nl = (size_t)ctx->p.n_layers + 1;
    const size_t need = (size_t)ctx->plan.n_chunks * ctx->p.n_cols * 4 * nl * 8;
    if (need > (size_t)HELIOS_STATIC_SCRATCH_BYTES) {
        snprintf(ctx->err, sizeof ctx->err, "helios_fluxes_static: this shape needs %zu bytes of partial sums, the "
                 "static scratch holds %zu (HELIOS_STATIC_SCRATCH_BYTES); use helios_fluxes", need,
                 (size_t)HELIOS_STATIC_SCRATCH_BYTES);
        return HELIOS_E_WORKSPACE;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail_cuda(ctx, "cudaGetDevice");
    if (dev != ctx->device) return fail(ctx, HELIOS_E_BADARG, "helios_fluxes_static: the context's device is not the current device");
    if (!ctx->static_scratch) return fail(ctx, HELIOS_E_CUDA, "helios_fluxes_static: cudaGetSymbolAddress failed at set-up");
    DevView v = ctx->v;                        // the context's own view (partial -> workspace) stays as it is
    v.partial = static_cast<double*>(ctx->static_scratch);
    v.spec_up_toa = nullptr;
    v.spec_dn_boa = nullptr;
    v.warm_now = 0;                            // one-shot evaluations are cold
    HX_LAUNCH(ctx, launch_clear_nonfinite(v, ctx->st));
    HX_LAUNCH(ctx, launch_flux(v, 0, ctx->st));            // no event pairs: creating one would allocate
    HX_LAUNCH(ctx, launch_reduce(v, 0, 0, 0.0, 0.0, ctx->st));
    const size_t fb = (size_t)ctx->p.n_cols * nl * 8;
    if (F_up) HX_CUDA(ctx, cudaMemcpyAsync(F_up, v.F_up, fb, cudaMemcpyDeviceToDevice, ctx->st));
    if (F_dn) HX_CUDA(ctx, cudaMemcpyAsync(F_dn, v.F_dn, fb, cudaMemcpyDeviceToDevice, ctx->st));
    return HELIOS_OK;
}

int helios_fluxes_host(helios_ctx* ctx, const double* T_host, double* F_up_host, double* F_dn_host)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const size_t tb = (size_t)ctx->p.n_cols * ctx->p.n_layers * 8;
    const size_t fb = (size_t)ctx->p.n_cols * (ctx->p.n_layers + 1) * 8;
    if (T_host) HX_CUDA(ctx, cudaMemcpyAsync(ctx->ws + ctx->plan.o_T, T_host, tb, cudaMemcpyHostToDevice, ctx->st));
    ctx->v.warm_now = 0;
    HX_LAUNCH(ctx, launch_clear_nonfinite(ctx->v, ctx->st));
    HX_LAUNCH(ctx, flux_launch(ctx, 0));
    HX_LAUNCH(ctx, launch_reduce(ctx->v, 0, 0, 0.0, 0.0, ctx->st));
    if (F_up_host) HX_CUDA(ctx, cudaMemcpyAsync(F_up_host, ctx->v.F_up, fb, cudaMemcpyDeviceToHost, ctx->st));
    if (F_dn_host) HX_CUDA(ctx, cudaMemcpyAsync(F_dn_host, ctx->v.F_dn, fb, cudaMemcpyDeviceToHost, ctx->st));
    const int r = check_flags(ctx);
    if (r != HELIOS_OK) return r;
    if (ctx->h_flags[1]) return fail(ctx, HELIOS_E_NONFINITE, "non-finite flux");
    return HELIOS_OK;
}

static int iterate_core(helios_ctx* ctx, int32_t max_iter, double tol_dT, double tol_flux, int32_t poll_every)
{
    if (max_iter < 0) return fail(ctx, HELIOS_E_BADARG, "max_iter < 0");
    if (poll_every <= 0) poll_every = 16;
    const bool has_tol = tol_dT > 0.0 || tol_flux > 0.0;
    ctx->v.warm_now = ctx->p.warm_start;       // RE steps start from the previous step's upward fluxes (S4)
    HX_LAUNCH(ctx, launch_clear_nonfinite(ctx->v, ctx->st));
    HX_LAUNCH(ctx, launch_count_running(ctx->v, ctx->st));   // columns flagged by an earlier call take part again
    // Launch-bound loops (small batches) replay a captured graph of poll_every iterations; the
    // per-launch event timing of helios_enable_timing needs individual launches.
    const bool use_graph = ctx->gst && !ctx->timing && max_iter >= poll_every;
    cudaStream_t run = ctx->st;
    int it = 0;
    if (use_graph) {
        const int rg = ensure_graph(ctx, poll_every, tol_dT, tol_flux);
        if (rg != HELIOS_OK) return rg;
        run = ctx->gst;
        HX_CUDA(ctx, cudaEventRecord(ctx->g_in, ctx->st));
        HX_CUDA(ctx, cudaStreamWaitEvent(run, ctx->g_in, 0));
        bool done = false;
        for (; it + poll_every <= max_iter && !done; it += poll_every) {
            HX_CUDA(ctx, cudaGraphLaunch(ctx->gexec, run));
            ctx->launches += 2 * poll_every;
            if (has_tol && it + poll_every < max_iter) {
                const int r = check_flags(ctx, run);
                if (r != HELIOS_OK) return r;
                if (ctx->h_flags[1]) return fail(ctx, HELIOS_E_NONFINITE, "non-finite temperature step");
                done = ctx->h_flags[0] == 0;
            }
        }
        if (done) it = max_iter;
    }
    for (; it < max_iter; ++it) {
        if (run == ctx->st) HX_LAUNCH(ctx, flux_launch(ctx, 1));
        else HX_LAUNCH(ctx, launch_flux(ctx->v, 1, run));
        HX_LAUNCH(ctx, launch_reduce(ctx->v, 1, 1, tol_dT, tol_flux, run));
        if (has_tol && ((it + 1) % poll_every == 0) && it + 1 < max_iter) {
            const int r = check_flags(ctx, run);
            if (r != HELIOS_OK) return r;
            if (ctx->h_flags[1]) return fail(ctx, HELIOS_E_NONFINITE, "non-finite temperature step");
            if (ctx->h_flags[0] == 0) break;
        }
    }
    const int r = check_flags(ctx, run);
    if (r != HELIOS_OK) return r;
    if (run != ctx->st) {
        HX_CUDA(ctx, cudaEventRecord(ctx->g_out, run));
        HX_CUDA(ctx, cudaStreamWaitEvent(ctx->st, ctx->g_out, 0));
    }
    if (ctx->h_flags[1]) return fail(ctx, HELIOS_E_NONFINITE, "non-finite temperature step");
    return HELIOS_OK;
}

int helios_iterate_re(helios_ctx* ctx, int32_t max_iter, double tol_dT, double tol_flux,
                      int32_t poll_every, double* T_out, int32_t* iters, int32_t* converged)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const int r = iterate_core(ctx, max_iter, tol_dT, tol_flux, poll_every);
    if (r != HELIOS_OK) return r;
    const size_t nc = ctx->p.n_cols, n = ctx->p.n_layers;
    if (T_out) HX_CUDA(ctx, cudaMemcpyAsync(T_out, ctx->v.T, nc * n * 8, cudaMemcpyDeviceToDevice, ctx->st));
    if (iters) HX_CUDA(ctx, cudaMemcpyAsync(iters, ctx->v.iters, nc * 4, cudaMemcpyDeviceToDevice, ctx->st));
    if (converged) HX_CUDA(ctx, cudaMemcpyAsync(converged, ctx->v.converged, nc * 4, cudaMemcpyDeviceToDevice, ctx->st));
    return HELIOS_OK;
}

int helios_iterate_re_host(helios_ctx* ctx, int32_t max_iter, double tol_dT, double tol_flux,
                           int32_t poll_every, double* T_host_inout, int32_t* iters_host,
                           int32_t* converged_host)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const size_t nc = ctx->p.n_cols, n = ctx->p.n_layers;
    if (T_host_inout) HX_CUDA(ctx, cudaMemcpyAsync(ctx->v.T, T_host_inout, nc * n * 8, cudaMemcpyHostToDevice, ctx->st));
    const int r = iterate_core(ctx, max_iter, tol_dT, tol_flux, poll_every);
    if (r != HELIOS_OK) return r;
    if (T_host_inout) HX_CUDA(ctx, cudaMemcpyAsync(T_host_inout, ctx->v.T, nc * n * 8, cudaMemcpyDeviceToHost, ctx->st));
    if (iters_host) HX_CUDA(ctx, cudaMemcpyAsync(iters_host, ctx->v.iters, nc * 4, cudaMemcpyDeviceToHost, ctx->st));
    if (converged_host) HX_CUDA(ctx, cudaMemcpyAsync(converged_host, ctx->v.converged, nc * 4, cudaMemcpyDeviceToHost, ctx->st));
    HX_CUDA(ctx, cudaStreamSynchronize(ctx->st));
    return HELIOS_OK;
}

int helios_get_re_state(helios_ctx* ctx, double* step_factor, int32_t* sign_hist, double* dT_last)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const size_t k = (size_t)ctx->p.n_cols * ctx->p.n_layers;
    if (step_factor) HX_CUDA(ctx, cudaMemcpyAsync(step_factor, ctx->v.step_factor, k * 8, cudaMemcpyDeviceToDevice, ctx->st));
    if (sign_hist) HX_CUDA(ctx, cudaMemcpyAsync(sign_hist, ctx->v.sign_hist, k * 4, cudaMemcpyDeviceToDevice, ctx->st));
    if (dT_last) HX_CUDA(ctx, cudaMemcpyAsync(dT_last, ctx->v.dT_last, k * 8, cudaMemcpyDeviceToDevice, ctx->st));
    return HELIOS_OK;
}

int helios_get_re_metrics(helios_ctx* ctx, double* max_dT, double* max_rel_dF, int32_t* nonfinite)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const size_t nc = ctx->p.n_cols;
    if (max_dT) HX_CUDA(ctx, cudaMemcpyAsync(max_dT, ctx->v.col_max_dT, nc * 8, cudaMemcpyDeviceToDevice, ctx->st));
    if (max_rel_dF) HX_CUDA(ctx, cudaMemcpyAsync(max_rel_dF, ctx->v.col_max_rel, nc * 8, cudaMemcpyDeviceToDevice, ctx->st));
    if (nonfinite) HX_CUDA(ctx, cudaMemcpyAsync(nonfinite, ctx->v.col_nonfinite, nc * 4, cudaMemcpyDeviceToDevice, ctx->st));
    return HELIOS_OK;
}

int helios_set_re_state(helios_ctx* ctx, const double* step_factor, const int32_t* sign_hist,
                        const int32_t* iters, const int32_t* converged)
{
    if (!ctx) return HELIOS_E_BADARG;
    if (!ctx->columns_set) return fail(ctx, HELIOS_E_NOTSETUP, "helios_set_columns has not been called");
    const size_t nc = ctx->p.n_cols, k = nc * ctx->p.n_layers;
    if (step_factor) HX_CUDA(ctx, cudaMemcpyAsync(ctx->v.step_factor, step_factor, k * 8, cudaMemcpyDeviceToDevice, ctx->st));
    if (sign_hist) HX_CUDA(ctx, cudaMemcpyAsync(ctx->v.sign_hist, sign_hist, k * 4, cudaMemcpyDeviceToDevice, ctx->st));
    if (iters) HX_CUDA(ctx, cudaMemcpyAsync(ctx->v.iters, iters, nc * 4, cudaMemcpyDeviceToDevice, ctx->st));
    if (converged) HX_CUDA(ctx, cudaMemcpyAsync(ctx->v.converged, converged, nc * 4, cudaMemcpyDeviceToDevice, ctx->st));
    HX_LAUNCH(ctx, launch_count_running(ctx->v, ctx->st));
    return HELIOS_OK;
}

int helios_get_fluxes(helios_ctx* ctx, double* F_up, double* F_dn)
{
    if (!ctx) return HELIOS_E_BADARG;
    const size_t fb = (size_t)ctx->p.n_cols * (ctx->p.n_layers + 1) * 8;
    if (F_up) HX_CUDA(ctx, cudaMemcpyAsync(F_up, ctx->v.F_up, fb, cudaMemcpyDeviceToDevice, ctx->st));
    if (F_dn) HX_CUDA(ctx, cudaMemcpyAsync(F_dn, ctx->v.F_dn, fb, cudaMemcpyDeviceToDevice, ctx->st));
    return HELIOS_OK;
}

int helios_enable_timing(helios_ctx* ctx, int32_t on)
{
    if (!ctx) return HELIOS_E_BADARG;
    ctx->timing = on != 0;
    return HELIOS_OK;
}

int helios_kernel_time_ms(helios_ctx* ctx, double* total_ms, int64_t* launches)
{
    if (!ctx || !total_ms || !launches) return HELIOS_E_BADARG;
    HX_CUDA(ctx, cudaStreamSynchronize(ctx->st));
    double sum = 0.0;
    for (size_t i = 0; i < ctx->ev_used; ++i) {
        float ms = 0.f;
        HX_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev[2 * i], ctx->ev[2 * i + 1]));
        sum += ms;
    }
    *total_ms = sum;
    *launches = (int64_t)ctx->ev_used;
    ctx->ev_used = 0;
    return HELIOS_OK;
}

int64_t helios_launch_count(const helios_ctx* ctx) { return ctx ? ctx->launches : 0; }

int helios_launch_shape(const helios_ctx* ctx, int32_t out[5])
{
    if (!ctx || !out) return HELIOS_E_BADARG;
    out[0] = ctx->p.n_cols;
    out[1] = ctx->plan.n_chunks;
    out[2] = 32 * ctx->plan.warps;
    out[3] = (int32_t)ctx->plan.smem;
    out[4] = ctx->plan.S;
    return HELIOS_OK;
}

double helios_measure_fma_peak(int32_t precision, void* cuda_stream)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return (double)HELIOS_E_CUDA; }
    if (precision != HELIOS_PREC_FP64 && precision != HELIOS_PREC_FP32) return (double)HELIOS_E_BADARG;
    return measure_fma_peak(precision, 0, reinterpret_cast<cudaStream_t>(cuda_stream));
}

double helios_measure_fma3_peak(int32_t precision, void* cuda_stream)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return (double)HELIOS_E_CUDA; }
    if (precision != HELIOS_PREC_FP64 && precision != HELIOS_PREC_FP32) return (double)HELIOS_E_BADARG;
    return measure_fma_peak(precision, 1, reinterpret_cast<cudaStream_t>(cuda_stream));
}

const char* helios_last_error(const helios_ctx* ctx) { return ctx ? ctx->err : g_noctx_err; }

void helios_destroy(helios_ctx* ctx)
{
    if (!ctx) return;
    if (ctx->h_flags) cudaFreeHost(ctx->h_flags);
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    if (ctx->gexec) cudaGraphExecDestroy(ctx->gexec);
    if (ctx->g_in) cudaEventDestroy(ctx->g_in);
    if (ctx->g_out) cudaEventDestroy(ctx->g_out);
    if (ctx->gst) cudaStreamDestroy(ctx->gst);
    delete ctx;
}

}  // extern "C"
