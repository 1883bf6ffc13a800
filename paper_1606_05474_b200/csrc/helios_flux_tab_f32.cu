// helios_flux_tab_f32.cu -- third variant of the ray kernel of helios_flux.cu: the benchmarked kernel plus the tabulated
// Planck function (planck_table_dT > 0, S15), fp32 ray arithmetic.  Product code (CUDA path, sm_100a);
// shares nothing with oracle/.
#define HX_FLUX_ALT 2
#define HX_FLUX_F32 1
#include "helios_flux.cu"
