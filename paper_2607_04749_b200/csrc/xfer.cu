// xfer.cu — metadata transfers that stay off the copy engines.
//
// The planning calls move a few hundred bytes to a few megabytes between host and device (device maps, pointer tables,
// piece tables, the plan totals).  As cudaMemcpyAsync these go through the DMA copy engines, where they queue behind
// whatever bulk transfers are already pending there (measured: with a host-resident pipeline uploading gigabytes, a
// 200-byte read-back of the plan totals waited 70 ms for the previous pass's downloads).  So:
//   host -> device, small : the bytes ride in the kernel's parameter block (write_small)
//   pinned host <-> device: a grid-stride copy kernel reads / writes the pinned buffer directly (copy_by_kernel);
//                           pinned memory is device-addressable at its host address
// Both are ordinary kernels on the caller's stream: they wait for nothing but that stream.  Used where the transfer is
// ordered with kernels of that stream anyway (device map and failure mask before the plan kernels, plan totals after
// them, pointer tables before the copy kernels, round records).  The layout tables are NOT moved this way: they are
// uploaded on a private stream while the copy kernels of a migration in flight fill the SMs, and there a DMA copy runs
// beside them where a copy kernel waits for them (measured: 0.16 ms -> 1.7 ms per layout pair on c2).
#include <cstring>
#include <mutex>
#include "etc_internal.h"

namespace etc {

constexpr int PARAM_BYTES = 3840;                    // kernel parameters are limited to 4 KB in total
struct ParamBlock { unsigned char b[PARAM_BYTES]; };

__global__ void __launch_bounds__(256) write_params_kernel(const __grid_constant__ ParamBlock p, unsigned char* __restrict__ dst, int n) {
  for (int i = threadIdx.x; i < n; i += blockDim.x) dst[i] = p.b[i];
}

__global__ void __launch_bounds__(256) copy16_kernel(uint4* __restrict__ dst, const uint4* __restrict__ src, size_t n16) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}
__global__ void __launch_bounds__(256) copy1_kernel(unsigned char* __restrict__ dst, const unsigned char* __restrict__ src, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

cudaError_t write_small(void* d_dst, const void* h_src, size_t bytes, cudaStream_t st) {
  const unsigned char* src = static_cast<const unsigned char*>(h_src);
  unsigned char* dst = static_cast<unsigned char*>(d_dst);
  for (size_t off = 0; off < bytes; off += PARAM_BYTES) {
    ParamBlock p;
    const int n = (int)(bytes - off < (size_t)PARAM_BYTES ? bytes - off : (size_t)PARAM_BYTES);
    memcpy(p.b, src + off, (size_t)n);
    write_params_kernel<<<1, 256, 0, st>>>(p, dst + off, n);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    count_launch();
  }
  return cudaSuccess;
}

cudaError_t copy_by_kernel(void* dst, const void* src, size_t bytes, cudaStream_t st) {
  if (bytes == 0) return cudaSuccess;
  const bool aligned = ((reinterpret_cast<uintptr_t>(dst) | reinterpret_cast<uintptr_t>(src) | bytes) & 15) == 0;
  if (aligned) {
    const size_t n16 = bytes / 16;
    const unsigned grid = (unsigned)((n16 + 255) / 256 < 1184 ? (n16 + 255) / 256 : 1184);     // <= 8 CTAs per SM
    copy16_kernel<<<grid, 256, 0, st>>>(static_cast<uint4*>(dst), static_cast<const uint4*>(src), n16);
  } else {
    const unsigned grid = (unsigned)((bytes + 255) / 256 < 1184 ? (bytes + 255) / 256 : 1184);
    copy1_kernel<<<grid, 256, 0, st>>>(static_cast<unsigned char*>(dst), static_cast<const unsigned char*>(src), bytes);
  }
  count_launch();
  return cudaGetLastError();
}


// grow-only pinned scratch for read-backs; hold pinned_scratch_mutex() from the call until the data has been copied out
static std::mutex g_scratch_mu;
static void* g_scratch = nullptr;
static size_t g_scratch_cap = 0;
std::mutex& pinned_scratch_mutex() { return g_scratch_mu; }
void* pinned_scratch(size_t bytes) {
  if (bytes > g_scratch_cap) {
    if (g_scratch) cudaFreeHost(g_scratch);
    g_scratch = nullptr; g_scratch_cap = 0;
    const size_t cap = bytes < (64u << 10) ? (64u << 10) : bytes + bytes / 2;
    if (cudaMallocHost(&g_scratch, cap) != cudaSuccess) { (void)cudaGetLastError(); g_scratch = nullptr; return nullptr; }
    g_scratch_cap = cap;
  }
  return g_scratch;
}

}  // namespace etc
