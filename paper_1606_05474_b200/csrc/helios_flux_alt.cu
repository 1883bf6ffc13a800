// helios_flux_alt.cu -- second instantiation of the ray kernel of helios_flux.cu: the one that also holds the
// exact pure-absorption limit (exact_absorption = 1, S13) and the single-scattering albedo per
// sublayer (helios_set_scattering, S14).  Product code (CUDA path, sm_100a); shares nothing with oracle/.
#define HX_FLUX_ALT 1
#include "helios_flux.cu"
