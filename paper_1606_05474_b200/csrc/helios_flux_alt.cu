// helios_flux_alt.cu -- second variant of the ray kernel of helios_flux.cu, fp64: the one that also holds the
// exact pure-absorption limit (exact_absorption = 1, S13) and the single-scattering albedo per
// sublayer (helios_set_scattering, S14).  Product code (CUDA path, sm_100a); shares nothing with oracle/.
#define HX_FLUX_ALT 1
#define HX_FLUX_F32 0
#include "helios_flux.cu"
