// cost.cu — (a2) cost matrix by integer index-range intersection (PAPER.md:106 c_ij = len(curr_i) - len(curr_i ∩ prev_j);
// :167-169 TP units and PP/TP merge are subsumed by intersecting index rectangles directly).
//
// One warp (or one CTA, when there are few cells) owns one matrix cell (new rank n, old device o): lanes walk n's pieces, look the matching (kind, tensor)
// group of o up in o's dense first-piece table, intersect rectangles and warp-reduce.  No atomics, so every cell is
// written exactly once and the result is order-independent.  Extra warps past the matrix compute need[] and hold[].
#include <algorithm>
#include <vector>
#include "etc_internal.h"

namespace etc {

__device__ __forceinline__ int64_t isect_elems(const Piece& a, const Piece& b) {
  const int r0 = max(a.r0, b.r0), r1 = min(a.r0 + a.nr, b.r0 + b.nr);
  const int c0 = max(a.c0, b.c0), c1 = min(a.c0 + a.nc, b.c0 + b.nc);
  return (r1 > r0 && c1 > c0) ? (int64_t)(r1 - r0) * (int64_t)(c1 - c0) : 0;
}

__device__ __forceinline__ int64_t warp_sum(int64_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

constexpr int COST_WARPS = 8;

// WPC = warps per job.  WPC = 1: eight jobs per CTA (many cells: 512 x 384 layouts).  WPC = 8: the whole CTA shares one
// job and reduces through shared memory (few cells: the piece lists are long compared with the cell count, so one
// warp per cell would leave most of the machine idle and serialise ~20 dependent loads per lane).
// A block of cells that can be non-zero: the devices of one new pipeline stage x the devices of one old stage that shares
// layers (or embeddings) with it.  base = cells of the blocks before this one.
struct StageBlock { int32_t n0, nn, o0, on; long long base; };

template <int WPC>
__global__ void __launch_bounds__(COST_WARPS * 32)
cost_matrix_kernel(DeviceTables oldT, DeviceTables newT, int P,
                   int64_t* __restrict__ overlap, int64_t* __restrict__ need, int64_t* __restrict__ hold,
                   const StageBlock* __restrict__ blocks, int n_blocks, long long block_cells) {
  __shared__ int64_t s_part[COST_WARPS];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int sub = wid % WPC;                                  // this warp's share of the job
  const long long job = ((long long)blockIdx.x * COST_WARPS + wid) / WPC;
  // with a block list (many devices: most cells pair different pipeline stages and are zero — the matrix was cleared, and
  // only the listed blocks get a warp), a job is a cell of one block; otherwise a cell of the whole matrix
  const long long cells = blocks ? block_cells : (long long)newT.n_dev * P;
  const int stride = 32 * WPC;
  int64_t acc = 0;
  int64_t* out = nullptr;
  if (job < cells) {
    int n, o;
    if (blocks) {
      int lo = 0, hi = n_blocks - 1;                            // the block whose cell range holds `job`
      while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (blocks[mid].base <= job) lo = mid; else hi = mid - 1; }
      const StageBlock b = blocks[lo];
      const long long local = job - b.base;
      n = b.n0 + (int)(local / b.on); o = b.o0 + (int)(local % b.on);
    } else {
      n = (int)(job / P); o = (int)(job % P);
    }
    out = overlap + (size_t)n * P + o;
    if (o < oldT.n_dev) {
      // early out: no logical tensor in common (different pipeline stages)
      bool common = false;
      for (int w = lane; w < newT.mask_words; w += 32)
        common |= (newT.ltmask[(size_t)n * newT.mask_words + w] & oldT.ltmask[(size_t)o * oldT.mask_words + w]) != 0;
      if (__any_sync(0xffffffffu, common)) {
        const int qb = newT.dev_start[n], qe = newT.dev_start[n + 1], oe = oldT.dev_start[o + 1];
        const int nT = newT.n_tensors;
        for (int i = qb + sub * 32 + lane; i < qe; i += stride) {
          const Piece q = newT.pieces[i];
          int j = oldT.first[(size_t)o * oldT.n_grp + q.grp];
          if (j < 0) continue;
          int64_t e = 0;
          for (; j < oe; ++j) {
            const Piece& p = oldT.pieces[j];
            if (p.grp != q.grp) break;
            e += isect_elems(q, p);
          }
          acc += e * newT.elem_bytes[q.grp / nT];
        }
      }
    }
  } else if (job < cells + newT.n_dev + P) {                  // need[n] / hold[o]: bytes of all pieces of one device
    const long long k = job - cells;
    const bool is_need = k < newT.n_dev;
    const int dev = is_need ? (int)k : (int)(k - newT.n_dev);
    const Piece* pieces = is_need ? newT.pieces : oldT.pieces;
    const int32_t* dev_start = is_need ? newT.dev_start : oldT.dev_start;
    const int n_dev = is_need ? newT.n_dev : oldT.n_dev, nT = newT.n_tensors;
    out = (is_need ? need : hold) + dev;
    if (dev < n_dev)
      for (int i = dev_start[dev] + sub * 32 + lane; i < dev_start[dev + 1]; i += stride) {
        const Piece& q = pieces[i];
        acc += (int64_t)q.nr * q.nc * newT.elem_bytes[q.grp / nT];
      }
  }
  acc = warp_sum(acc);
  if (WPC == 1) {
    if (lane == 0 && out) *out = acc;
  } else {
    if (lane == 0) s_part[wid] = acc;
    __syncthreads();
    if (threadIdx.x == 0 && out) {
      int64_t t = 0;
#pragma unroll
      for (int k = 0; k < COST_WARPS; ++k) t += s_part[k];
      *out = t;
    }
  }
}

}  // namespace etc

using namespace etc;

static bool same_model(const etc_layout* a, const etc_layout* b) {
  const etc_model_desc &x = a->model, &y = b->model;
  return x.style == y.style && x.n_layers == y.n_layers && x.hidden == y.hidden && x.n_q_heads == y.n_q_heads &&
         x.n_kv_heads == y.n_kv_heads && x.head_dim == y.head_dim && x.ffn_hidden == y.ffn_hidden &&
         x.vocab == y.vocab && x.max_pos == y.max_pos && x.tied_embeddings == y.tied_embeddings &&
         x.param_dtype == y.param_dtype && x.kinds == y.kinds && x.qkv_order == y.qkv_order;
}
bool etc_same_model(const etc_layout* a, const etc_layout* b) { return same_model(a, b); }

extern "C" etc_status etc_cost_matrix(const etc_layout* old_l, const etc_layout* new_l, int64_t* d_overlap,
                                      int64_t* d_need, int64_t* d_hold, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!old_l || !new_l || !d_overlap || !d_need || !d_hold) return ETC_ERR_INVALID_ARG;
  if (!same_model(old_l, new_l)) return ETC_ERR_MISMATCH;
  const int P = old_l->t.n_dev > new_l->t.n_dev ? old_l->t.n_dev : new_l->t.n_dev;
  ETC_CUDA_TRY(layout_use(old_l, (cudaStream_t)stream));
  ETC_CUDA_TRY(layout_use(new_l, (cudaStream_t)stream));
  const long long jobs = (long long)new_l->t.n_dev * P + new_l->t.n_dev + P;
  cudaStream_t st = (cudaStream_t)stream;
  if (jobs <= 8192) {
    cost_matrix_kernel<COST_WARPS><<<(unsigned)jobs, COST_WARPS * 32, 0, st>>>(
        old_l->t, new_l->t, P, d_overlap, d_need, d_hold, nullptr, 0, 0);
  } else {
    // Many devices: list the (new stage, old stage) blocks that can overlap — stages whose layer ranges intersect, and the
    // first / last stages among themselves (embeddings, final norm, output layer, the tied replica) — clear the matrix and
    // give warps to those blocks only.  Device ids are stage-major (r + tp*(d + dp*s)), so a stage is a contiguous range.
    const std::vector<int32_t>&fo = old_l->stage_first, &fn = new_l->stage_first;
    const int ppo = old_l->t.pp, ppn = new_l->t.pp;
    const int dso = old_l->t.tp * old_l->t.dp, dsn = new_l->t.tp * new_l->t.dp;
    std::vector<StageBlock> blocks;
    long long bc = 0;
    for (int sn = 0; sn < ppn; ++sn)
      for (int so = 0; so < ppo; ++so) {
        const bool layers = std::max(fn[sn], fo[so]) < std::min(fn[sn + 1], fo[so + 1]);
        const bool ends = (sn == 0 || sn == ppn - 1) && (so == 0 || so == ppo - 1);
        if (!layers && !ends) continue;
        blocks.push_back(StageBlock{sn * dsn, dsn, so * dso, dso, bc});
        bc += (long long)dsn * dso;
      }
    if (bc * 2 <= (long long)new_l->t.n_dev * P && !blocks.empty()) {
      StageBlock* d_blocks = nullptr;
      ETC_CUDA_TRY(cudaMallocAsync(&d_blocks, sizeof(StageBlock) * blocks.size(), st));
      cudaError_t e = write_small(d_blocks, blocks.data(), sizeof(StageBlock) * blocks.size(), st);
      if (e == cudaSuccess) e = cudaMemsetAsync(d_overlap, 0, sizeof(int64_t) * (size_t)new_l->t.n_dev * P, st);
      if (e == cudaSuccess) {
        const long long bjobs = bc + new_l->t.n_dev + P;
        cost_matrix_kernel<1><<<(unsigned)((bjobs + COST_WARPS - 1) / COST_WARPS), COST_WARPS * 32, 0, st>>>(
            old_l->t, new_l->t, P, d_overlap, d_need, d_hold, d_blocks, (int)blocks.size(), bc);
        e = cudaGetLastError();
      }
      cudaFreeAsync(d_blocks, st);
      ETC_CUDA_TRY(e);
    } else {
      cost_matrix_kernel<1><<<(unsigned)((jobs + COST_WARPS - 1) / COST_WARPS), COST_WARPS * 32, 0, st>>>(
          old_l->t, new_l->t, P, d_overlap, d_need, d_hold, nullptr, 0, 0);
    }
  }
  ETC_CUDA_TRY(cudaGetLastError());
  count_launch();
  return ETC_OK;
}

// (f4) reading A26: a failed old device holds nothing — zero its column of the overlap matrix and its
// hold entry, so the sketch keeps nothing "local" on it.
namespace etc {
__global__ void mask_failed_kernel(int64_t* __restrict__ overlap, int64_t* __restrict__ hold, int n_new, int n_old, int P,
                                   const uint8_t* __restrict__ failed) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)(n_new + 1) * n_old) return;
  const int o = (int)(i % n_old), n = (int)(i / n_old);
  if (!failed[o]) return;
  if (n < n_new) overlap[(size_t)n * P + o] = 0; else if (hold) hold[o] = 0;
}
}  // namespace etc

extern "C" etc_status etc_mask_failed(int64_t* d_overlap, int64_t* d_hold, int32_t n_new, int32_t n_old, int32_t P,
                                      const uint8_t* d_failed, void* stream) {
  etc::clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!d_overlap || !d_failed || n_new < 1 || n_old < 1 || P < n_old || P < n_new) return ETC_ERR_INVALID_ARG;
  const long long total = (long long)(n_new + 1) * n_old;
  etc::mask_failed_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream>>>(d_overlap, d_hold, n_new,
                                                                                              n_old, P, d_failed);
  ETC_CUDA_TRY(cudaGetLastError());
  etc::count_launch();
  return ETC_OK;
}

// The paper's own treatment of the DP dimension (reading A5): processes under different DP ranks
// are isolated, "the difference between the workloads [is] infinite" — a cross-DP cell keeps nothing local.
namespace etc {
__global__ void mask_cross_dp_kernel(int64_t* __restrict__ overlap, int n_new, int n_old, int P, int tp_o, int dp_o,
                                     int tp_n, int dp_n) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)n_new * n_old) return;
  const int o = (int)(i % n_old), n = (int)(i / n_old);
  if ((o / tp_o) % dp_o != (n / tp_n) % dp_n) overlap[(size_t)n * P + o] = 0;      // device id = r + tp*(d + dp*s)
}
}  // namespace etc

extern "C" etc_status etc_mask_cross_dp(const etc_layout* old_l, const etc_layout* new_l, int64_t* d_overlap, void* stream) {
  etc::clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!old_l || !new_l || !d_overlap) return ETC_ERR_INVALID_ARG;
  if (!same_model(old_l, new_l)) return ETC_ERR_MISMATCH;
  const int n_old = old_l->t.n_dev, n_new = new_l->t.n_dev, P = n_old > n_new ? n_old : n_new;
  const long long total = (long long)n_new * n_old;
  etc::mask_cross_dp_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
      d_overlap, n_new, n_old, P, old_l->t.tp, old_l->t.dp, new_l->t.tp, new_l->t.dp);
  ETC_CUDA_TRY(cudaGetLastError());
  etc::count_launch();
  return ETC_OK;
}
