// rp_to_q.cu -- S1, Eq. 9:  g(Re,q) = sum_Rp g(Re,Rp) w_p e^{i q.Rp}.
//
// The paper runs this as one ZGEMV per q: every q re-reads all 16 Nb^2 Nm Ne Np bytes of g,
// 0.5 flop/byte, HBM-bound.  Here NQ q-points share one streaming pass over g (a skinny GEMM,
// [rows x Np] . [Np x NQ]): g is read once per batch with coalesced 16-byte loads, NQ complex accumulators
// live in registers, and the phase columns are broadcast from shared memory.  HBM roofline: 16*rows*Np bytes
// read + 16*rows*NQ bytes written per launch.
#include "common.cuh"

namespace epw {

template <int NQ>
__global__ void __launch_bounds__(256) rp_to_q_kernel(const c128 *__restrict__ g, int64_t rows, int np,
                                                      const c128 *__restrict__ Pq, c128 *__restrict__ g1) {
  extern __shared__ double2 sP[];  // [np][NQ]
  for (int e = threadIdx.x; e < np * NQ; e += blockDim.x) {
    const int ip = e / NQ, iq = e - ip * NQ;
    sP[e] = Pq[(int64_t)iq * np + ip];
  }
  __syncthreads();
  const int64_t row = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (row >= rows) return;
  c128 acc[NQ];
#pragma unroll
  for (int iq = 0; iq < NQ; iq++) acc[iq] = cmake(0.0, 0.0);
  const c128 *col = g + row;
  int ip = 0;
  constexpr int U = 8;  // independent 16-byte loads in flight per thread
  for (; ip + U <= np; ip += U) {
    c128 v[U];
#pragma unroll
    for (int u = 0; u < U; u++) v[u] = __ldcs(col + (int64_t)(ip + u) * rows);
#pragma unroll
    for (int u = 0; u < U; u++) {
#pragma unroll
      for (int iq = 0; iq < NQ; iq++) cfma(acc[iq], v[u], sP[(ip + u) * NQ + iq]);
    }
  }
  for (; ip < np; ip++) {
    const c128 v = __ldcs(col + (int64_t)ip * rows);
#pragma unroll
    for (int iq = 0; iq < NQ; iq++) cfma(acc[iq], v, sP[ip * NQ + iq]);
  }
#pragma unroll
  for (int iq = 0; iq < NQ; iq++) g1[(int64_t)iq * rows + row] = acc[iq];
}

template <int NQ>
static cudaError_t launch_nq(const c128 *g, int64_t rows, int np, const c128 *Pq, c128 *g1, cudaStream_t st) {
  const size_t smem = sizeof(double2) * (size_t)np * NQ;
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(rp_to_q_kernel<NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  rp_to_q_kernel<NQ><<<(unsigned)ceil_div(rows, 256), 256, smem, st>>>(g, rows, np, Pq, g1);
  return cudaGetLastError();
}

cudaError_t launch_rp_to_q(const c128 *g, int64_t rows, int np, const c128 *Pq, int nq, c128 *g1, cudaStream_t st) {
  switch (nq) {
    case 1: return launch_nq<1>(g, rows, np, Pq, g1, st);
    case 2: return launch_nq<2>(g, rows, np, Pq, g1, st);
    case 3: return launch_nq<3>(g, rows, np, Pq, g1, st);
    case 4: return launch_nq<4>(g, rows, np, Pq, g1, st);
    case 5: return launch_nq<5>(g, rows, np, Pq, g1, st);
    case 6: return launch_nq<6>(g, rows, np, Pq, g1, st);
    case 7: return launch_nq<7>(g, rows, np, Pq, g1, st);
    case 8: return launch_nq<8>(g, rows, np, Pq, g1, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace epw
