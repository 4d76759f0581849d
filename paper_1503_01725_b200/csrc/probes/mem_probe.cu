// mem_probe.cu — measurement probes, NOT part of libpslmc or its ABI: the two random-access ceilings the transport
// kernels are compared with in bench.py and profiles/ (DESIGN.md §5).  Built into libpslmc_probe.so.
//   probe_red64    nothing but int64 scoring atomics (RED.64) on pseudo-random voxels of a grid of nvox voxels
//   probe_gather32 nothing but dependent-free random 4-byte gathers from a table of n_words words (the packed phantom)
// Both: DEVICE buffer from the caller, ms_out HOST float[2] = (milliseconds by CUDA events, operations issued).
#include <cstdint>
#include <cuda_runtime.h>

namespace {
constexpr int kThreads = 256;

__device__ __forceinline__ unsigned pick(unsigned &x, unsigned n) {
  x = x * 1664525u + 1013904223u;
  return (unsigned)(((unsigned long long)(x ^ (x >> 15)) * n) >> 32);
}
__global__ void k_red64(unsigned long long *acc, unsigned nvox, unsigned per_thread, unsigned seed) {
  unsigned x = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + seed;
  for (unsigned i = 0; i < per_thread; ++i) atomicAdd(acc + pick(x, nvox), 1ull + i);
}
__global__ void k_gather32(const unsigned *tab, unsigned n, unsigned per_thread, unsigned seed, unsigned *sink) {
  unsigned x = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + seed, s = 0;
#pragma unroll 4
  for (unsigned i = 0; i < per_thread; ++i) s += __ldg(tab + pick(x, n));       // independent loads: 4 in flight per thread
  if (s == 0xdeadbeefu) *sink = s;
}
template <typename F>
int timed(F launch, unsigned threads, unsigned per_thread, float *ms_out) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -4;
  launch(16u, 0u);                                             // warm-up
  cudaEventRecord(e0);
  launch(per_thread, 1u);
  cudaEventRecord(e1);
  if (cudaEventSynchronize(e1) != cudaSuccess) return -4;
  cudaEventElapsedTime(ms_out, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  ms_out[1] = (float)((double)per_thread * threads);
  return cudaGetLastError() == cudaSuccess ? 0 : -4;
}
unsigned grid_blocks() { int dev = 0, sms = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); return (unsigned)sms * 8u; }
}  // namespace

extern "C" int probe_red64(int64_t *acc, uint64_t nvox, uint64_t n_ops, uint64_t seed, float *ms_out) {
  if (!acc || !ms_out || nvox == 0 || nvox >= 0x7fffffffull || n_ops == 0) return -1;
  const unsigned blocks = grid_blocks(), threads = blocks * kThreads, per = (unsigned)(n_ops / threads > 0 ? n_ops / threads : 1);
  return timed([&](unsigned p, unsigned s) { k_red64<<<blocks, kThreads>>>((unsigned long long *)acc, (unsigned)nvox, p, (unsigned)seed + s); }, threads, per, ms_out);
}
extern "C" int probe_gather32(const uint32_t *tab, uint64_t n_words, uint64_t n_ops, uint64_t seed, float *ms_out) {
  if (!tab || !ms_out || n_words == 0 || n_words >= 0x7fffffffull || n_ops == 0) return -1;
  unsigned *sink = nullptr; if (cudaMalloc(&sink, 4) != cudaSuccess) return -4;
  const unsigned blocks = grid_blocks(), threads = blocks * kThreads, per = (unsigned)(n_ops / threads > 0 ? n_ops / threads : 1);
  int rc = timed([&](unsigned p, unsigned s) { k_gather32<<<blocks, kThreads>>>(tab, (unsigned)n_words, p, (unsigned)seed + s, sink); }, threads, per, ms_out);
  cudaFree(sink);
  return rc;
}
