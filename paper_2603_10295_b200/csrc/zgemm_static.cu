// zgemm_static.cu -- epw_zgemm_noalloc: the dense complex FP64 contraction of epw_zgemm (pack A, pack B, DMMA kernel)
// for callers that are not allowed to allocate device memory.
//
// Who that is: code that runs inside somebody else's memory budget or latency budget -- a solver that has handed all of
// HBM to its own pool allocator (a cudaMalloc from a library would fail or fragment it), a real-time / in-situ loop in
// which cudaMalloc and cudaFree are forbidden because both synchronise the whole device, and hosts whose policy is that
// a plug-in library never grows the process's device footprint after it has been loaded.  epw_zgemm itself allocates
// the two packed operands with cudaMalloc on every call and frees them after a stream synchronise; this file does the
// same three launches with the packed operands in a fixed array that is part of the library image.
//
// The array lives in this translation unit only.  In HOST code its name is a stand-in symbol, not a device address, so
// the host side asks the runtime for the real address once per device (cudaGetSymbolAddress with that device current)
// and hands that pointer to the launchers.
#include <cstdio>
#include <mutex>

#include "common.cuh"

namespace epw {
namespace {

// 1,024 chunks of 16 KB = 16 MiB, held by every GPU that loads the library until the process exits.
constexpr int64_t NOALLOC_CHUNKS = EPW_ZGEMM_NOALLOC_SCRATCH_BYTES / (sizeof(double) * GEMM_CHUNK);
static_assert(NOALLOC_CHUNKS * sizeof(double) * GEMM_CHUNK == EPW_ZGEMM_NOALLOC_SCRATCH_BYTES, "whole chunks only");

static __device__ __align__(256) double zgemm_noalloc_scratch[NOALLOC_CHUNKS * GEMM_CHUNK];

constexpr int MAX_DEVICES = 64;
std::mutex g_addr_mu;
double *g_addr_of[MAX_DEVICES] = {nullptr};   // device address of the array on each device ordinal, once looked up

void say(char *errbuf, size_t errbuf_len, const char *fmt, long long a = 0, long long b = 0, long long c = 0) {
  if (errbuf && errbuf_len) snprintf(errbuf, errbuf_len, fmt, a, b, c);
}

// Device address of zgemm_noalloc_scratch on the CURRENT device.  The first call on a device is the set-up: it makes the
// runtime load this module on that device (which is when the 16 MiB come into existence there) and asks for the address.
int scratch_on_current_device(double **out, char *errbuf, size_t errbuf_len) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) {
    say(errbuf, errbuf_len, "epw_zgemm_noalloc: no current CUDA device (or ordinal %lld >= 64)", dev);
    return EPW_ECUDA;
  }
  std::lock_guard<std::mutex> lock(g_addr_mu);
  if (!g_addr_of[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, zgemm_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      if (errbuf && errbuf_len)
        snprintf(errbuf, errbuf_len, "epw_zgemm_noalloc: cudaGetSymbolAddress of the static scratch failed on device %d: %s",
                 dev, cudaGetErrorString(e));
      return EPW_ECUDA;
    }
    g_addr_of[dev] = static_cast<double *>(p);
  }
  *out = g_addr_of[dev];
  return EPW_OK;
}

}  // namespace
}  // namespace epw

using namespace epw;

extern "C" int epw_zgemm_noalloc(const void *A, const void *B, void *C, int64_t M, int32_t N, int32_t K, int64_t ldc,
                                 void *cuda_stream, char *errbuf, size_t errbuf_len) {
  if (errbuf && errbuf_len) errbuf[0] = '\0';
  if (!A || !B || !C || M <= 0 || N <= 0 || K <= 0 || ldc < N) {
    say(errbuf, errbuf_len, "epw_zgemm_noalloc: null pointer, non-positive size or ldc < N");
    return EPW_EINVAL;
  }
  // packed sizes, exactly as epw_zgemm lays them out: A' = MT x KB chunks, B' = NT x KB chunks of 16 KB
  const int64_t KB = ceil_div(2 * (int64_t)K, GEMM_BK);
  const int64_t NT = ceil_div(2 * (int64_t)N, GEMM_BN);
  const int64_t MT = ceil_div(M, GEMM_BM);
  const int64_t chunks_a = MT * KB, chunks_b = NT * KB;
  if (MT > NOALLOC_CHUNKS || NT > NOALLOC_CHUNKS || chunks_a + chunks_b > NOALLOC_CHUNKS) {
    say(errbuf, errbuf_len,
        "epw_zgemm_noalloc: the packed operands need %lld chunks of 16 KB, the static scratch holds %lld "
        "(ceil(M/128)*ceil(K/8) + ceil(N/64)*ceil(K/8) <= %lld); split the product or use epw_zgemm",
        (long long)(chunks_a + chunks_b), (long long)NOALLOC_CHUNKS, (long long)NOALLOC_CHUNKS);
    return EPW_EUNSUPPORTED;
  }
  double *scratch = nullptr;
  const int rc = scratch_on_current_device(&scratch, errbuf, errbuf_len);
  if (rc != EPW_OK) return rc;
  double *Ap = scratch, *Bp = scratch + chunks_a * GEMM_CHUNK;   // both 16 KB aligned
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  // Nothing has to be cleared first although the array keeps whatever the previous call left in it: the two pack kernels
  // write every double of every chunk the product reads, the zero padding of ragged tiles included.
  cudaError_t e = launch_pack_a_generic(reinterpret_cast<const c128 *>(A), M, K, Ap, st);
  if (e == cudaSuccess) e = launch_pack_b_generic(reinterpret_cast<const c128 *>(B), K, N, Bp, st);
  if (e == cudaSuccess)
    e = launch_zgemm_dmma(Ap, Bp, reinterpret_cast<c128 *>(C), M, N, (int)KB, ldc, device_sm_count(), st);
  if (e != cudaSuccess) {
    if (errbuf && errbuf_len) snprintf(errbuf, errbuf_len, "epw_zgemm_noalloc: launch failed: %s", cudaGetErrorString(e));
    return e == cudaErrorInvalidValue ? EPW_EINVAL : EPW_ECUDA;
  }
  return EPW_OK;
}
