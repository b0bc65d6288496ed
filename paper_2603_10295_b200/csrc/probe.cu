// probe.cu -- roofline denominators measured on the device in use:
// FP64 tensor peak (DMMA m8n8k4 issue loop), plain FP64 FMA peak, HBM read and copy bandwidth.
// MEASURED_PEAKS.json carries no FP64 figure, so bench.py reports the DMMA number from here next to it.
#include <algorithm>

#include "common.cuh"

namespace epw {

__global__ void __launch_bounds__(256) probe_dmma_kernel(double *out, int iters) {
  double c[16][2];
#pragma unroll
  for (int i = 0; i < 16; i++) c[i][0] = c[i][1] = 0.0;
  const double a = threadIdx.x * 1e-3, b = 1.0 + threadIdx.x * 1e-4;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[i][0]), "+d"(c[i][1])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += c[i][0] + c[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) probe_dfma_kernel(double *out, int iters, double a, double b) {
  double acc[16];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = fma(acc[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += acc[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void probe_read_kernel(const double2 *__restrict__ in, double *out, size_t n) {
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  double s = 0.0;
  for (; i < n; i += stride) {
    const double2 v = in[i];
    s += v.x + v.y;
  }
  if (s == 1.2345e300) out[0] = s;
}
__global__ void probe_copy_kernel(const double2 *__restrict__ in, double2 *__restrict__ out, size_t n) {
  size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; i < n; i += stride) out[i] = in[i];
}

template <class F>
static float best_ms(F f, int reps) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  f();
  cudaDeviceSynchronize();
  float best = 1e30f;
  for (int r = 0; r < reps; r++) {
    cudaEventRecord(e0);
    f();
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    best = std::min(best, ms);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return best;
}

int probe_peaks(int device, double *out4) {
  if (cudaSetDevice(device) != cudaSuccess) return EPW_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return EPW_ECUDA;
  const int nsm = prop.multiProcessorCount;
  double *out = nullptr;
  const size_t n = (size_t)1 << 27;  // 2 GiB of double2 per buffer
  double2 *a = nullptr, *b = nullptr;
  if (cudaMalloc(&out, sizeof(double) * nsm * 2 * 256) != cudaSuccess) return EPW_ENOMEM;
  if (cudaMalloc(&a, n * 16) != cudaSuccess || cudaMalloc(&b, n * 16) != cudaSuccess) {
    cudaFree(out); cudaFree(a); cudaFree(b);
    return EPW_ENOMEM;
  }
  cudaMemset(a, 1, n * 16);
  cudaMemset(b, 0, n * 16);
  const int iters = 20000, grid = nsm * 2;
  float ms = best_ms([&] { probe_dmma_kernel<<<grid, 256>>>(out, iters); }, 3);
  out4[0] = 2.0 * 256 * 16 * (double)iters * 8.0 * grid / ms * 1e-9;
  ms = best_ms([&] { probe_dfma_kernel<<<grid, 256>>>(out, iters, 1.0000001, 1e-9); }, 3);
  out4[1] = 2.0 * 16 * (double)iters * 256.0 * grid / ms * 1e-9;
  ms = best_ms([&] { probe_read_kernel<<<nsm * 16, 512>>>(a, out, n); }, 5);
  out4[2] = (double)n * 16 / ms * 1e-6;
  ms = best_ms([&] { probe_copy_kernel<<<nsm * 32, 512>>>(a, b, n); }, 5);
  out4[3] = 2.0 * (double)n * 16 / ms * 1e-6;
  const cudaError_t err = cudaDeviceSynchronize();
  cudaFree(out); cudaFree(a); cudaFree(b);
  return err == cudaSuccess ? EPW_OK : EPW_ECUDA;
}

}  // namespace epw
