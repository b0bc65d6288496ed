// grid_fused_nb13.cu -- instantiates the kernels of grid_fused.cuh for Nb = 13 .. 16 (see grid_fused.cu)
#include "grid_fused.cuh"

namespace epw {

cudaError_t launch_gf_nb13(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st) {
  switch (nb) {
    case 13: return launch_gf<13>(p, num_sms, st);
    case 14: return launch_gf<14>(p, num_sms, st);
    case 15: return launch_gf<15>(p, num_sms, st);
    case 16: return launch_gf<16>(p, num_sms, st);
    default: return cudaErrorInvalidConfiguration;
  }
}

}  // namespace epw
