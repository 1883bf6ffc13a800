// helios_flux_dispatch.cu -- routes the ray-kernel calls of helios_api.cu to the translation unit that holds
// the kernel: helios_flux.cu is compiled once per (variant, arithmetic, lanes per ray), see build.py.
// Product code; shares nothing with oracle/.
#include "helios_internal.h"

namespace hx {

#define HX_DECL_UNIT(tag)                                                        \
    int flux_configure##tag(int S, int iso, size_t smem_bytes);                  \
    int launch_flux##tag(const DevView& v, int respect_converged, cudaStream_t st);
#define HX_DECL_LPR(vp)  HX_DECL_UNIT(vp##_l8) HX_DECL_UNIT(vp##_l16) HX_DECL_UNIT(vp##_l32)
HX_DECL_LPR(_main_f64) HX_DECL_LPR(_main_f32) HX_DECL_LPR(_alt_f64) HX_DECL_LPR(_alt_f32) HX_DECL_LPR(_tab_f64) HX_DECL_LPR(_tab_f32)
#define HX_DECL_SMEM(tag) size_t flux_smem##tag(int S, int warps, int iso);
HX_DECL_SMEM(_main_f64_l8) HX_DECL_SMEM(_main_f64_l16) HX_DECL_SMEM(_main_f64_l32)
HX_DECL_SMEM(_main_f32_l8) HX_DECL_SMEM(_main_f32_l16) HX_DECL_SMEM(_main_f32_l32)

// calls fn<variant><arithmetic><lpr>(args)
#define HX_BY_LPR(fn, vp, lpr, ...) \
    ((lpr) == 8 ? fn##vp##_l8(__VA_ARGS__) : (lpr) == 16 ? fn##vp##_l16(__VA_ARGS__) : fn##vp##_l32(__VA_ARGS__))

// per warp two (bin id, up, down) entries: the spectrum shares of the partial bins at the two ends of its unit run
size_t flux_spec_smem_bytes(int warps, int unit_split)
{
    return unit_split ? (size_t)warps * 6 * sizeof(double) : 0;
}

size_t flux_smem_bytes(int lpr, int S, int warps, int iso, int precision)
{
    if (precision == HELIOS_PREC_FP32) return HX_BY_LPR(flux_smem, _main_f32, lpr, S, warps, iso);
    return HX_BY_LPR(flux_smem, _main_f64, lpr, S, warps, iso);
}

int flux_configure(int lpr, int S, int iso, int precision, size_t smem_bytes)
{
    if (precision == HELIOS_PREC_FP32)
        return (HX_BY_LPR(flux_configure, _alt_f32, lpr, S, iso, smem_bytes) == 0 &&
                HX_BY_LPR(flux_configure, _tab_f32, lpr, S, iso, smem_bytes) == 0 &&
                HX_BY_LPR(flux_configure, _main_f32, lpr, S, iso, smem_bytes) == 0) ? 0 : -1;
    return (HX_BY_LPR(flux_configure, _alt_f64, lpr, S, iso, smem_bytes) == 0 &&
            HX_BY_LPR(flux_configure, _tab_f64, lpr, S, iso, smem_bytes) == 0 &&
            HX_BY_LPR(flux_configure, _main_f64, lpr, S, iso, smem_bytes) == 0) ? 0 : -1;
}

int launch_flux(const DevView& v, int respect_converged, cudaStream_t st)
{
    const bool alt = v.exact || v.kscat;   // exact limit / albedo per sublayer
    const bool tab = v.ptab != nullptr || v.tt_dlog > 0.0;    // tabulated Planck / transmission function
    if (v.precision == HELIOS_PREC_FP32)
        return alt ? HX_BY_LPR(launch_flux, _alt_f32, v.lpr, v, respect_converged, st)
                   : tab ? HX_BY_LPR(launch_flux, _tab_f32, v.lpr, v, respect_converged, st)
                         : HX_BY_LPR(launch_flux, _main_f32, v.lpr, v, respect_converged, st);
    return alt ? HX_BY_LPR(launch_flux, _alt_f64, v.lpr, v, respect_converged, st)
               : tab ? HX_BY_LPR(launch_flux, _tab_f64, v.lpr, v, respect_converged, st)
                     : HX_BY_LPR(launch_flux, _main_f64, v.lpr, v, respect_converged, st);
}

}  // namespace hx
