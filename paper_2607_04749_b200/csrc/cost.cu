// cost.cu — (a2) cost matrix by integer index-range intersection (PAPER.md:106 c_ij = len(curr_i) - len(curr_i ∩ prev_j);
// :167-169 TP units and PP/TP merge are subsumed by intersecting index rectangles directly).
//
// One warp owns one matrix cell (new rank n, old device o): lanes walk n's pieces, look the matching (kind, tensor)
// group of o up in o's dense first-piece table, intersect rectangles and warp-reduce.  No atomics, so every cell is
// written exactly once and the result is order-independent.  Extra warps past the matrix compute need[] and hold[].
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

__global__ void __launch_bounds__(COST_WARPS * 32)
cost_matrix_kernel(DeviceTables oldT, DeviceTables newT, int P,
                   int64_t* __restrict__ overlap, int64_t* __restrict__ need, int64_t* __restrict__ hold) {
  const int lane = threadIdx.x & 31;
  const long long warp = (long long)blockIdx.x * COST_WARPS + (threadIdx.x >> 5);
  const long long cells = (long long)newT.n_dev * P;
  if (warp < cells) {
    const int n = (int)(warp / P), o = (int)(warp % P);
    int64_t acc = 0;
    if (o < oldT.n_dev) {
      // early out: no logical tensor in common (different pipeline stages)
      bool common = false;
      for (int w = lane; w < newT.mask_words; w += 32)
        common |= (newT.ltmask[(size_t)n * newT.mask_words + w] & oldT.ltmask[(size_t)o * oldT.mask_words + w]) != 0;
      if (__any_sync(0xffffffffu, common)) {
        const int qb = newT.dev_start[n], qe = newT.dev_start[n + 1], oe = oldT.dev_start[o + 1];
        const int nT = newT.n_tensors;
        for (int i = qb + lane; i < qe; i += 32) {
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
    acc = warp_sum(acc);
    if (lane == 0) overlap[warp] = acc;
    return;
  }
  // need[n] / hold[o]: bytes of all pieces of one device
  const long long job = warp - cells;
  if (job < newT.n_dev + P) {
    const bool is_need = job < newT.n_dev;
    const DeviceTables& T = is_need ? newT : oldT;
    const int dev = is_need ? (int)job : (int)(job - newT.n_dev);
    int64_t acc = 0;
    if (dev < T.n_dev)
      for (int i = T.dev_start[dev] + lane; i < T.dev_start[dev + 1]; i += 32) {
        const Piece& q = T.pieces[i];
        acc += (int64_t)q.nr * q.nc * T.elem_bytes[q.grp / T.n_tensors];
      }
    acc = warp_sum(acc);
    if (lane == 0) (is_need ? need : hold)[dev] = acc;
  }
}

}  // namespace etc

using namespace etc;

static bool same_model(const etc_layout* a, const etc_layout* b) {
  const etc_model_desc &x = a->model, &y = b->model;
  return x.style == y.style && x.n_layers == y.n_layers && x.hidden == y.hidden && x.n_q_heads == y.n_q_heads &&
         x.n_kv_heads == y.n_kv_heads && x.head_dim == y.head_dim && x.ffn_hidden == y.ffn_hidden &&
         x.vocab == y.vocab && x.max_pos == y.max_pos && x.tied_embeddings == y.tied_embeddings &&
         x.param_dtype == y.param_dtype && x.kinds == y.kinds;
}
bool etc_same_model(const etc_layout* a, const etc_layout* b) { return same_model(a, b); }

extern "C" etc_status etc_cost_matrix(const etc_layout* old_l, const etc_layout* new_l, int64_t* d_overlap,
                                      int64_t* d_need, int64_t* d_hold, void* stream) {
  clear_error_detail();
  if (!old_l || !new_l || !d_overlap || !d_need || !d_hold) return ETC_ERR_INVALID_ARG;
  if (!same_model(old_l, new_l)) return ETC_ERR_MISMATCH;
  const int P = old_l->t.n_dev > new_l->t.n_dev ? old_l->t.n_dev : new_l->t.n_dev;
  const long long warps = (long long)new_l->t.n_dev * P + new_l->t.n_dev + P;
  const unsigned grid = (unsigned)((warps + COST_WARPS - 1) / COST_WARPS);
  cost_matrix_kernel<<<grid, COST_WARPS * 32, 0, (cudaStream_t)stream>>>(old_l->t, new_l->t, P, d_overlap, d_need,
                                                                          d_hold);
  ETC_CUDA_TRY(cudaGetLastError());
  count_launch();
  return ETC_OK;
}
