// grid_fused_nb9.cu -- instantiates the kernels of grid_fused.cuh for Nb = 9 .. 12 (see grid_fused.cu)
#include "grid_fused.cuh"

namespace epw {

cudaError_t launch_gf_nb9(int nb, const GridFusedParams &p, int num_sms, cudaStream_t st) {
  switch (nb) {
    case 9: return launch_gf<9>(p, num_sms, st);
    case 10: return launch_gf<10>(p, num_sms, st);
    case 11: return launch_gf<11>(p, num_sms, st);
    case 12: return launch_gf<12>(p, num_sms, st);
    default: return cudaErrorInvalidConfiguration;
  }
}

}  // namespace epw
