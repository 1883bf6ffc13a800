// helios_flux_alt_f32.cu -- second variant of the ray kernel of helios_flux.cu (see helios_flux_alt.cu),
// fp32 ray arithmetic.  Product code (CUDA path, sm_100a); shares nothing with oracle/.
#define HX_FLUX_ALT 1
#define HX_FLUX_F32 1
#include "helios_flux.cu"
