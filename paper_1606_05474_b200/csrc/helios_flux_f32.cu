// helios_flux_f32.cu -- the ray kernel of helios_flux.cu with fp32 ray arithmetic (HELIOS_PREC_FP32).
// Product code (CUDA path, sm_100a); shares nothing with oracle/.
#define HX_FLUX_ALT 0
#define HX_FLUX_F32 1
#include "helios_flux.cu"
