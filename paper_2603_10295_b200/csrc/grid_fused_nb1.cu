// grid_fused_nb1.cu -- instantiates the kernels of grid_fused.cuh for Nb = 1 .. 4 (see grid_fused.cu)
#include "grid_fused.cuh"

namespace epw {

cudaError_t launch_gf_nb1(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st) {
  switch (nb) {
    case 1: return launch_gf<1>(p, num_sms, st);
    case 2: return launch_gf<2>(p, num_sms, st);
    case 3: return launch_gf<3>(p, num_sms, st);
    case 4: return launch_gf<4>(p, num_sms, st);
    default: return cudaErrorInvalidConfiguration;
  }
}

}  // namespace epw
