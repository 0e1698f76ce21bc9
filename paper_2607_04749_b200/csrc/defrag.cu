// defrag.cu — (f1) virtual rank allocator: Algorithm 2 "Placement-Aware Remapping" (§III-E) on the
// device, composed with the migration sketch into ONE final device_map (communication coalescing, PAPER.md:224, :269:
// "if (1) sends the workload w from device i to device k, and (2) sends w from k to j, the execution engine coalesces
// these two instructions into sending w from i to j").  Because etc_plan_create takes the final map, the second hop
// never exists: every element goes from its source straight to the device that finally hosts its rank.
//
// The listing of Algorithm 2 is garbled (reading A23); this follows the prose PAPER.md:220-222:
//   occupancy   (lines 1-9):  p2c[device] = curr rank on it or -1 (dropped / idle).  Idle devices in ascending order are
//                             paired with occupied devices in descending order until the two meet; the process on the
//                             occupied device moves to the idle one.
//   efficiency  (lines 10-20): target placement = curr rank k on device k (n consecutive ranks per node, so TP groups sit
//                             inside a node); every device of a fragmented node whose load differs from its target gets
//                             an operator <target rank, current load>.
// Integer work on <= P devices: one CTA, block-wide prefix sums (warp shuffles) for the ordered idle / occupied / operator
// lists.  Everything is enqueued on the caller's stream; no host synchronisation.
#include "etc_internal.h"

namespace etc {

constexpr int DF_THREADS = 1024;

// exclusive block scan of one int per thread; returns the exclusive prefix, total via reference.  All threads call it.
__device__ __forceinline__ int block_excl_scan(int v, int& total, int* s_warp /* [33] */) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  __syncthreads();                                   // s_warp may still be read from the previous call
  if (lane == 31) s_warp[wid] = x;
  __syncthreads();
  if (wid == 0) {
    int w = s_warp[lane], y = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int z = __shfl_up_sync(0xffffffffu, y, o); if (lane >= o) y += z; }
    s_warp[lane] = y - w;
    if (lane == 31) s_warp[32] = y;
  }
  __syncthreads();
  total = s_warp[32];
  return s_warp[wid] + x - v;
}

// ws: p2c [P] | idle_list [P] | occ_list [P]
__global__ void __launch_bounds__(DF_THREADS)
defrag_kernel(const int32_t* __restrict__ map_in, int pw, int cw, int P, int n_per_node, int mode,
              int32_t* __restrict__ map_out, int32_t* __restrict__ ops, int32_t* __restrict__ n_ops,
              int32_t* __restrict__ ws) {
  __shared__ int s_warp[33];
  __shared__ int s_bad, s_cnt;
  int32_t* p2c = ws; int32_t* idle_list = ws + P; int32_t* occ_list = ws + 2 * (size_t)P;
  const int tid = threadIdx.x;
  if (tid == 0) { s_bad = 0; s_cnt = 0; }
  for (int i = tid; i < P; i += DF_THREADS) p2c[i] = -1;
  __syncthreads();
  // invert the sketch: p2c[physical device] = curr rank
  for (int r = tid; r < cw; r += DF_THREADS) {
    const int dev = map_in[r];
    if (dev < 0 || dev >= P) s_bad = 1;
    else if (atomicCAS(&p2c[dev], -1, r) != -1) s_bad = 1;
  }
  __syncthreads();
  if (s_bad) {                                       // not an injective map into [0,P): report, write nothing useful
    for (int r = tid; r < cw; r += DF_THREADS) map_out[r] = -1;
    if (tid < 2) n_ops[tid] = -1;
    return;
  }
  for (int r = tid; r < cw; r += DF_THREADS) map_out[r] = map_in[r];
  int n_occ_ops = 0, n_eff_ops = 0;

  if (mode & ETC_DEFRAG_OCCUPANCY) {
    // lines 6-7: idle devices in order, occupied devices in reverse order
    int base_idle = 0, base_occ = 0;
    for (int t0 = 0; t0 < P; t0 += DF_THREADS) {
      const int i = t0 + tid, j = P - 1 - i;         // i ascending for idle, j descending for occupied
      const int f_idle = (i < P && p2c[i] == -1) ? 1 : 0;
      const int f_occ = (i < P && p2c[j] != -1) ? 1 : 0;
      int tot_i, tot_o;
      const int e_i = block_excl_scan(f_idle, tot_i, s_warp);
      const int e_o = block_excl_scan(f_occ, tot_o, s_warp);
      if (f_idle) idle_list[base_idle + e_i] = i;
      if (f_occ) occ_list[base_occ + e_o] = j;
      base_idle += tot_i; base_occ += tot_o;
    }
    __syncthreads();
    // lines 8-9: pair until the iterators meet (idle ascending, occupied descending => the condition is monotone in k)
    const int m = min(base_idle, base_occ);
    int mine = 0;
    for (int k = tid; k < m; k += DF_THREADS) {
      const int i = idle_list[k], o = occ_list[k];
      if (i < o) {
        const int rank = p2c[o];
        if (ops) { ops[2 * k] = i; ops[2 * k + 1] = o; }
        map_out[rank] = i;                           // coalesced: the rank lands on device i in one hop
        p2c[i] = rank; p2c[o] = -1;                  // idle and occupied sets are disjoint: no conflicts
        ++mine;
      }
    }
    if (mine) atomicAdd(&s_cnt, mine);
    __syncthreads();
    n_occ_ops = s_cnt;
    __syncthreads();
  }

  if (mode & ETC_DEFRAG_EFFICIENCY) {
    // lines 12-20: target = rank k on device k; a node is fragmented iff some device's load differs from its target,
    // and it contributes exactly those devices.  n_per_node only groups the comparison (line 16).
    int32_t* eops = ops ? ops + 2 * (size_t)cw : nullptr;
    int base = 0;
    for (int t0 = 0; t0 < cw; t0 += DF_THREADS) {
      const int k = t0 + tid;
      const int load = k < cw ? p2c[k] : -2;
      const int f = (k < cw && load != k) ? 1 : 0;
      int tot;
      const int e = block_excl_scan(f, tot, s_warp);
      if (f) {
        if (eops) { eops[2 * (base + e)] = k; eops[2 * (base + e) + 1] = load; }
        map_out[k] = k;
      }
      base += tot;
    }
    n_eff_ops = base;
  }
  (void)pw; (void)n_per_node;
  if (tid == 0) { n_ops[0] = n_occ_ops; n_ops[1] = n_eff_ops; }
}

}  // namespace etc

using namespace etc;

extern "C" etc_status etc_defrag(const int32_t* d_device_map, int32_t pw, int32_t cw, int32_t devices_per_node,
                                 int32_t mode, int32_t* d_out_map, int32_t* d_ops, int32_t* d_n_ops, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!d_device_map || !d_out_map || !d_n_ops) return ETC_ERR_INVALID_ARG;
  if (pw < 1 || cw < 1 || devices_per_node < 1) return ETC_ERR_INVALID_ARG;
  if (mode < ETC_DEFRAG_OCCUPANCY || mode > ETC_DEFRAG_BOTH) return ETC_ERR_INVALID_ARG;
  if (d_out_map == d_device_map) return ETC_ERR_INVALID_ARG;
  const int P = pw > cw ? pw : cw;
  cudaStream_t st = (cudaStream_t)stream;
  int32_t* ws = nullptr;
  ETC_CUDA_TRY(cudaMallocAsync(&ws, sizeof(int32_t) * 3 * (size_t)P, st));
  defrag_kernel<<<1, DF_THREADS, 0, st>>>(d_device_map, pw, cw, P, devices_per_node, mode, d_out_map, d_ops, d_n_ops, ws);
  cudaError_t e = cudaGetLastError();
  cudaFreeAsync(ws, st);
  if (e != cudaSuccess) { set_error_detail("defrag_kernel", e); return ETC_ERR_CUDA; }
  count_launch();
  return ETC_OK;
}
