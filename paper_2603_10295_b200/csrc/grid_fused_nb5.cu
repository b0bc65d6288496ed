// grid_fused_nb5.cu -- instantiates the kernels of grid_fused.cuh for Nb = 5 .. 8 (see grid_fused.cu)
#include "grid_fused.cuh"

namespace epw {

cudaError_t launch_gf_nb5(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st) {
  switch (nb) {
    case 5: return launch_gf<5>(p, num_sms, st);
    case 6: return launch_gf<6>(p, num_sms, st);
    case 7: return launch_gf<7>(p, num_sms, st);
    case 8: return launch_gf<8>(p, num_sms, st);
    default: return cudaErrorInvalidConfiguration;
  }
}

}  // namespace epw
