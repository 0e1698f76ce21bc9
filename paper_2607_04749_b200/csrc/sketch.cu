// sketch.cu — (a3) migration sketch: pair current ranks with previous devices so that the most bytes stay in place
// (PAPER.md:110-132 assignment problem, Eq. 1-4; :134-163 Algorithm 1).  Objective (reading A4):
//   device_map = argmax over injective pi:[0,n_new)->[0,P) of sum_n overlap[n][pi(n)].
// Two device-side searches, both single-CTA (the problem is a few hundred rows: latency-bound integer work):
//   * exhaustive: every injective map enumerated by its mixed-radix index (P <= 8: at most 40 320 maps);
//   * Hungarian:  shortest augmenting paths with dual potentials on the rectangular matrix (rows <= columns, so no
//     zero padding is needed: padded rows of Algorithm 1 line 3 would cost 0 on every column and are dropped again by
//     lines 6-8).  One thread per column, block-wide arg-min per Dijkstra step.
#include <cstdio>
#include "etc_internal.h"

namespace etc {

constexpr int SK_THREADS = 1024;
constexpr int64_t SK_INF = (int64_t)1 << 62;
constexpr int64_t SK_UNSOLVED = -2;                 // sketch_tight_kernel -> sketch_hungarian_kernel: "no certificate, go on"

// ---------------------------------------------------------------------------------------------- exhaustive
__global__ void __launch_bounds__(SK_THREADS)
sketch_exhaustive_kernel(const int64_t* __restrict__ overlap, int N, int P, const uint8_t* __restrict__ avail,
                         int32_t* __restrict__ device_map, int64_t* __restrict__ local_bytes) {
  __shared__ int64_t ov[64];
  __shared__ int64_t s_val[32];
  __shared__ int s_idx[32];
  __shared__ uint32_t s_avail;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid < N * P) ov[tid] = overlap[tid];
  if (tid == 0) {
    uint32_t m = 0;
    for (int j = 0; j < P; ++j) if (!avail || avail[j]) m |= 1u << j;
    s_avail = m;
  }
  __syncthreads();
  int total = 1;
  for (int n = 0; n < N; ++n) total *= (P - n);
  const uint32_t all = (1u << P) - 1u, av = s_avail;

  int64_t best = -1; int best_idx = 0x7fffffff;
  for (int idx = tid; idx < total; idx += SK_THREADS) {
    int rem = idx; uint32_t used = 0; int64_t sum = 0;
    for (int n = 0; n < N; ++n) {
      const int radix = P - n, digit = rem % radix; rem /= radix;
      const int c = __fns(~used & all, 0, digit + 1);      // the digit-th still unused column
      used |= 1u << c; sum += ov[n * P + c];
    }
    if ((used & ~av) == 0 && sum > best) { best = sum; best_idx = idx; }   // idx ascending: ties keep the smallest
  }
  // block arg-max, ties -> smallest index (deterministic)
  auto better = [](int64_t v, int i, int64_t bv, int bi) { return v > bv || (v == bv && i < bi); };
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const int64_t v = __shfl_xor_sync(0xffffffffu, best, o); const int i = __shfl_xor_sync(0xffffffffu, best_idx, o);
    if (better(v, i, best, best_idx)) { best = v; best_idx = i; }
  }
  if (lane == 0) { s_val[wid] = best; s_idx[wid] = best_idx; }
  __syncthreads();
  if (wid == 0) {
    best = s_val[lane]; best_idx = s_idx[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const int64_t v = __shfl_xor_sync(0xffffffffu, best, o); const int i = __shfl_xor_sync(0xffffffffu, best_idx, o);
      if (better(v, i, best, best_idx)) { best = v; best_idx = i; }
    }
    if (lane == 0) {
      if (best < 0) {                                           // no feasible map
        for (int n = 0; n < N; ++n) device_map[n] = -1;
        *local_bytes = -1;
      } else {
        int rem = best_idx; uint32_t used = 0;
        for (int n = 0; n < N; ++n) {
          const int radix = P - n, digit = rem % radix; rem /= radix;
          const int c = __fns(~used & all, 0, digit + 1);
          used |= 1u << c; device_map[n] = c;
        }
        *local_bytes = best;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------- row-maximum certificate
// sum_n max_o overlap[n][o] bounds every sketch from above.  In the overlap matrices of real reconfigurations most rows
// have their maximum on a column no other row wants (or on one of several equal replicas, DP groups of the old layout), so
// a matching that gives EVERY row one of its maximal columns often exists — and any such matching is optimal.  This
// kernel looks for one greedily and, if it finds it, is done in a few microseconds where the O(k^3) search takes hundreds
// (512 -> 384 devices: 0.29 ms).  If it does not, it says so and sketch_hungarian_kernel runs as before: the fast path
// can only ever return an optimum.
//   1. (sketch_rowmax_kernel, one warp per row over the whole machine) the row maximum over the usable columns and its
//      first TK columns ("tight" columns); then one CTA (sketch_tight_kernel):
//   2. rows with a positive maximum claim a tight column (lowest row wins a contested one), rows with the fewest tight
//      columns first;
//   3. rows whose maximum is 0 overlap nothing anywhere: they take the columns left over, in order;
//   4. everyone placed -> device_map, local_bytes = the bound; else local_bytes = SK_UNSOLVED.
constexpr int TK = 4;                               // tight columns remembered per row
constexpr int TIGHT_MAX = 1024;                     // rows / columns the fast path handles (shared memory)
constexpr int RM_WARPS = 8;

// step 1, over the whole machine: one warp per row.  cnt[n] = tight columns found (capped at TK), -1 if the row's maximum is
// 0, -2 if the row has no usable column.
__global__ void __launch_bounds__(RM_WARPS * 32)
sketch_rowmax_kernel(const int64_t* __restrict__ overlap, int N, int P, const uint8_t* __restrict__ avail,
                     int64_t* __restrict__ rowmax, int32_t* __restrict__ cnt, int32_t* __restrict__ tight) {
  const int lane = threadIdx.x & 31, n = blockIdx.x * RM_WARPS + (threadIdx.x >> 5);
  if (n >= N) return;
  const int64_t* row = overlap + (size_t)n * P;
  int64_t m = -1;
#pragma unroll 8
  for (int j = lane; j < P; j += 32) { const int64_t x = row[j]; if (!avail || avail[j]) m = max(m, x); }   // loads first
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  int c = m < 0 ? -2 : (m == 0 ? -1 : 0);
  if (m > 0) {
    for (int j0 = 0; j0 < P && c < TK; j0 += 32) {
      const int j = j0 + lane;
      const bool t = j < P && (!avail || avail[j]) && row[j] == m;
      const unsigned mask = __ballot_sync(0xffffffffu, t);
      const int r = c + __popc(mask & ((1u << lane) - 1u));
      if (t && r < TK) tight[n * TK + r] = j;
      c += __popc(mask);
    }
    c = min(c, TK);
  }
  if (lane == 0) { cnt[n] = c; rowmax[n] = m; }
}

__global__ void __launch_bounds__(SK_THREADS)
sketch_tight_kernel(int N, int P, const uint8_t* __restrict__ avail, const int64_t* __restrict__ rowmax,
                    const int32_t* __restrict__ cnt_g, const int32_t* __restrict__ tight_g,
                    int32_t* __restrict__ device_map, int64_t* __restrict__ local_bytes) {
  __shared__ int32_t tight[TIGHT_MAX * TK];         // later reused: [0,P) free columns, [P, P+N) zero rows
  __shared__ int32_t cnt[TIGHT_MAX];                // tight columns of row n (capped at TK); -1: the row's maximum is 0
  __shared__ int32_t match[TIGHT_MAX];              // row -> column or -1
  __shared__ int32_t owner[TIGHT_MAX];              // column -> row, -1 free, -2 unusable
  __shared__ int32_t prop[TIGHT_MAX];               // column -> lowest row proposing to it
  __shared__ int64_t s_sum[32];
  __shared__ int32_t s_scan[33];
  __shared__ int s_bad;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid == 0) s_bad = 0;
  __syncthreads();
  for (int j = tid; j < P; j += SK_THREADS) { owner[j] = (!avail || avail[j]) ? -1 : -2; prop[j] = 0x7fffffff; }
  int64_t bound = 0;
  for (int n = tid; n < N; n += SK_THREADS) {
    match[n] = -1;
    const int c = cnt_g[n];
    cnt[n] = c;
    if (c == -2) s_bad = 1;                                      // a row with no usable column: infeasible, the search says so
    if (c > 0) bound += rowmax[n];
  }
  for (int i = tid; i < N * TK; i += SK_THREADS) tight[i] = tight_g[i];   // entries beyond cnt[n] are never read
  __syncthreads();
  // 2. claim tight columns, the most constrained rows first.  Deterministic: in every step the unmatched rows propose to
  // their next candidate and the LOWEST row wins a contested column (atomicMin), so the map does not depend on timing.
  for (int pass = 1; pass <= TK; ++pass) {
    for (int k = 0; k < pass; ++k) {
      for (int n = tid; n < N; n += SK_THREADS) {
        if (cnt[n] != pass || match[n] >= 0) continue;
        const int j = tight[n * TK + (k + n) % pass];            // spread rows that tie on the same columns
        if (owner[j] == -1) atomicMin(&prop[j], n);
      }
      __syncthreads();
      for (int n = tid; n < N; n += SK_THREADS) {
        if (cnt[n] != pass || match[n] >= 0) continue;
        const int j = tight[n * TK + (k + n) % pass];
        if (owner[j] == -1 && prop[j] == n) { owner[j] = n; match[n] = j; }
      }
      __syncthreads();
    }
    for (int n = tid; n < N; n += SK_THREADS) if (cnt[n] == pass && match[n] < 0) s_bad = 1;
    __syncthreads();
  }
  const bool bad = s_bad != 0;
  __syncthreads();
  if (!bad) {
    // 3. zero rows take the leftover columns: i-th zero row <-> i-th free column (compaction by block scans)
    int32_t* freec = tight; int32_t* zrow = tight + P;
    int n_free = 0, n_zero = 0;
    for (int pass = 0; pass < 2; ++pass) {
      const int L = pass == 0 ? P : N;
      int base = 0;
      for (int b0 = 0; b0 < L; b0 += SK_THREADS) {
        const int i = b0 + tid;
        const bool f = i < L && (pass == 0 ? owner[i] == -1 : cnt[i] == -1);
        const unsigned mask = __ballot_sync(0xffffffffu, f);
        if (lane == 0) s_scan[wid] = __popc(mask);
        __syncthreads();
        if (wid == 0) {
          int x = s_scan[lane], y = x;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) { const int z = __shfl_up_sync(0xffffffffu, y, o); if (lane >= o) y += z; }
          s_scan[lane] = y - x;
          if (lane == 31) s_scan[32] = y;
        }
        __syncthreads();
        if (f) (pass == 0 ? freec : zrow)[base + s_scan[wid] + __popc(mask & ((1u << lane) - 1u))] = i;
        base += s_scan[32];
        __syncthreads();
      }
      if (pass == 0) n_free = base; else n_zero = base;
    }
    if (n_zero > n_free) { if (tid == 0) s_bad = 1; }
    else for (int i = tid; i < n_zero; i += SK_THREADS) match[zrow[i]] = freec[i];
    __syncthreads();
  }
  if (s_bad) { if (tid == 0) *local_bytes = SK_UNSOLVED; return; }
  // 4. every row sits on one of its maximal columns: optimal
  for (int n = tid; n < N; n += SK_THREADS) device_map[n] = match[n];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) bound += __shfl_xor_sync(0xffffffffu, bound, o);
  if (lane == 0) s_sum[wid] = bound;
  __syncthreads();
  if (wid == 0) {
    int64_t t = s_sum[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) *local_bytes = t;
  }
}

// ---------------------------------------------------------------------------------------------- Hungarian
// Shortest augmenting path with potentials (the O(k^3) method Algorithm 1 calls through SciPy, ref [39]).
// cost(i,j) = -overlap[i][j]; columns masked by `avail` are never entered.  Per-column state lives in registers
// (CPT columns per thread), row potentials / matching / back-pointers in shared memory.
// The block is sized to the matrix: T threads x CPT columns per thread >= P (fewer warps = cheaper barriers and a
// shorter second reduction level); row i+1 is prefetched into registers while row i is being matched, so the first
// Dijkstra step of every augmentation — in a structured overlap matrix usually the only one — waits for no load.

struct ArgMin { int64_t v; int j; int matched; };
__device__ __forceinline__ bool argmin_less(const ArgMin& a, const ArgMin& b) {
  if (a.v != b.v) return a.v < b.v;
  if (a.matched != b.matched) return a.matched < b.matched;     // prefer a free column: the path ends at once
  return a.j < b.j;
}
// Warp arg-min of (v, matched, lane) in a handful of instructions instead of five rounds of four shuffles: the 64-bit
// minimum is two redux.sync ops (signed high word, then unsigned low word among the lanes that tie on the high word),
// the tie-break (a free column first, then the lowest lane) two ballots, and one shuffle fetches the winner's column.
__device__ __forceinline__ ArgMin warp_argmin(const ArgMin& a) {
  const int hi = (int)(a.v >> 32);
  const int mh = __reduce_min_sync(0xffffffffu, hi);
  const unsigned lo = hi == mh ? (unsigned)(a.v & 0xffffffffll) : 0xffffffffu;
  const unsigned ml = __reduce_min_sync(0xffffffffu, lo);
  const bool win = hi == mh && lo == ml;
  const unsigned m_all = __ballot_sync(0xffffffffu, win), m_free = __ballot_sync(0xffffffffu, win && !a.matched);
  const int src = __ffs(m_free ? m_free : m_all) - 1;
  ArgMin r;
  r.v = (int64_t)(((uint64_t)(uint32_t)mh << 32) | ml);
  r.j = __shfl_sync(0xffffffffu, a.j, src);
  r.matched = m_free ? 0 : 1;
  return r;
}

template <int SK_T, int SK_CPT>
__global__ void __launch_bounds__(SK_T)
sketch_hungarian_kernel(const int64_t* __restrict__ overlap, int N, int P, const uint8_t* __restrict__ avail,
                        int32_t* __restrict__ device_map, int64_t* __restrict__ local_bytes, int after_tight) {
  constexpr int SK_THREADS = SK_T, SK_NW = SK_T / 32;
  if (after_tight && *local_bytes != SK_UNSOLVED) return;      // sketch_tight_kernel found an optimum (uniform: one word)
  extern __shared__ __align__(16) unsigned char smem_raw[];
  int64_t* u = reinterpret_cast<int64_t*>(smem_raw);            // [N] row potentials
  int32_t* rowof = reinterpret_cast<int32_t*>(u + N);           // [P] column -> matched row or -1
  int32_t* way = rowof + P;                                     // [P] previous column on the alternating path
  __shared__ int64_t s_v[32]; __shared__ int s_j[32]; __shared__ int s_m[32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;

  int64_t v[SK_CPT], minv[SK_CPT]; bool used[SK_CPT], usable[SK_CPT];
#pragma unroll
  for (int c = 0; c < SK_CPT; ++c) {
    const int j = tid + c * SK_THREADS;
    v[c] = 0; usable[c] = j < P && (!avail || avail[j]);
    if (j < P) { rowof[j] = -1; way[j] = -1; }
  }
  for (int i = tid; i < N; i += SK_THREADS) u[i] = 0;
  __syncthreads();

  int64_t ahead[SK_CPT], row_i[SK_CPT];                         // row i+1 (in flight) and row i of the matrix
#pragma unroll
  for (int c = 0; c < SK_CPT; ++c) { const int j = tid + c * SK_THREADS; ahead[c] = j < P ? overlap[j] : 0; }

  bool fail = false;                                            // uniform across the block
  for (int i = 0; i < N; ++i) {
#pragma unroll
    for (int c = 0; c < SK_CPT; ++c) {
      const int j = tid + c * SK_THREADS;
      minv[c] = SK_INF; used[c] = !usable[c];
      row_i[c] = ahead[c];
      if (i + 1 < N && j < P) ahead[c] = overlap[(size_t)(i + 1) * P + j];
    }
    int i0 = i, j0 = -1;
    while (true) {
      // relax the edges of row i0, then block-wide arg-min of minv over the columns not yet on the tree
      const int64_t ui0 = u[i0];
      ArgMin best{SK_INF, 0x7fffffff, 1};
#pragma unroll
      for (int c = 0; c < SK_CPT; ++c) {
        const int j = tid + c * SK_THREADS;
        if (!used[c]) {
          const int64_t cur = -(j0 < 0 ? row_i[c] : overlap[(size_t)i0 * P + j]) - ui0 - v[c];
          if (cur < minv[c]) { minv[c] = cur; way[j] = j0; }
          ArgMin a{minv[c], j, rowof[j] >= 0 ? 1 : 0};
          if (argmin_less(a, best)) best = a;
        }
      }
      best = warp_argmin(best);
      if (lane == 0) { s_v[wid] = best.v; s_j[wid] = best.j; s_m[wid] = best.matched; }
      __syncthreads();
      best = warp_argmin(lane < SK_NW ? ArgMin{s_v[lane], s_j[lane], s_m[lane]} : ArgMin{SK_INF, 0x7fffffff, 1});
      if (best.v >= SK_INF) { fail = true; break; }                       // no column left: infeasible
      const int64_t delta = best.v; const int j1 = best.j;
      // dual update: tree rows gain delta, tree columns lose delta, the rest get closer by delta
      if (tid == 0) u[i] += delta;
#pragma unroll
      for (int c = 0; c < SK_CPT; ++c) {
        const int j = tid + c * SK_THREADS;
        if (j < P && usable[c]) {
          if (used[c]) { u[rowof[j]] += delta; v[c] -= delta; }
          else minv[c] -= delta;
          if (j == j1) used[c] = true;
        }
      }
      j0 = j1; i0 = rowof[j1];
      __syncthreads();
      if (i0 < 0) break;
    }
    if (fail) break;
    if (tid == 0) {                                                       // augment along the alternating path
      int j = j0;
      while (j >= 0) { const int jp = way[j]; rowof[j] = jp >= 0 ? rowof[jp] : i; j = jp; }
    }
    __syncthreads();
  }

  __syncthreads();
  if (fail) {
    for (int n = tid; n < N; n += SK_THREADS) device_map[n] = -1;
    if (tid == 0) *local_bytes = -1;
    return;
  }
  int64_t acc = 0;
#pragma unroll
  for (int c = 0; c < SK_CPT; ++c) {
    const int j = tid + c * SK_THREADS;
    if (j < P && rowof[j] >= 0) { device_map[rowof[j]] = j; acc += overlap[(size_t)rowof[j] * P + j]; }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  __syncthreads();
  if (lane == 0) s_v[wid] = acc;
  __syncthreads();
  if (wid == 0) {
    acc = lane < SK_NW ? s_v[lane] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) *local_bytes = acc;
  }
}

// Same algorithm for P <= 32: one warp, lane j owns column j, the matrix sits in shared memory, and every step is a
// handful of shuffles — no block barrier, no global-memory latency inside the Dijkstra loop.
__global__ void __launch_bounds__(32)
sketch_hungarian_warp_kernel(const int64_t* __restrict__ overlap, int N, int P, const uint8_t* __restrict__ avail,
                             int32_t* __restrict__ device_map, int64_t* __restrict__ local_bytes) {
  __shared__ int64_t ov[32 * 32];
  __shared__ int32_t way[32];
  __shared__ int64_t u[32];                   // row potentials
  const int lane = threadIdx.x;
  for (int i = lane; i < N * P; i += 32) ov[i] = overlap[i];
  u[lane] = 0;
  __syncwarp();
  const bool usable = lane < P && (!avail || avail[lane]);
  int64_t v = 0;                              // potential of column `lane`
  int rowof = -1;                             // row matched to column `lane`
  bool fail = false;
  for (int i = 0; i < N && !fail; ++i) {
    int64_t minv = SK_INF; bool used = !usable;
    int i0 = i, j0 = -1;
    while (true) {
      const int64_t ui0 = u[i0];
      ArgMin best{SK_INF, 0x7fffffff, 1};
      if (!used) {
        const int64_t cur = -ov[i0 * P + lane] - ui0 - v;
        if (cur < minv) { minv = cur; way[lane] = j0; }
        best = ArgMin{minv, lane, rowof >= 0 ? 1 : 0};
      }
      best = warp_argmin(best);
      if (best.v >= SK_INF) { fail = true; break; }
      const int64_t delta = best.v; const int j1 = best.j;
      // dual update: tree rows (the root i and the rows matched to tree columns) gain delta, tree columns lose it
      __syncwarp();
      if (lane == 0) u[i] += delta;
      if (usable) { if (used) { u[rowof] += delta; v -= delta; } else minv -= delta; if (lane == j1) used = true; }
      __syncwarp();
      j0 = j1; i0 = __shfl_sync(0xffffffffu, rowof, j1);
      if (i0 < 0) break;
    }
    if (fail) break;
    __syncwarp();
    // augment along the alternating path (every lane walks it; lane j updates its own column)
    int j = j0;
    while (j >= 0) {
      const int jp = way[j];
      const int r = jp >= 0 ? __shfl_sync(0xffffffffu, rowof, jp) : i;
      if (lane == j) rowof = r;
      j = jp;
    }
    __syncwarp();
  }
  if (fail) {
    if (lane < N) device_map[lane] = -1;
    if (lane == 0) *local_bytes = -1;
    return;
  }
  int64_t acc = 0;
  if (lane < P && rowof >= 0) { device_map[rowof] = lane; acc = ov[rowof * P + lane]; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) *local_bytes = acc;
}

}  // namespace etc

using namespace etc;

extern "C" etc_status etc_sketch(const int64_t* d_overlap, int32_t n_new, int32_t P, const uint8_t* d_avail,
                                 int32_t method, int32_t* d_device_map, int64_t* d_local_bytes, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!d_overlap || !d_device_map || !d_local_bytes || n_new < 1 || P < n_new) return ETC_ERR_INVALID_ARG;
  if (method == ETC_SKETCH_AUTO) method = ETC_SKETCH_HUNGARIAN;   // measured: faster than enumeration even at P = 8
  cudaStream_t st = (cudaStream_t)stream;
  if (method == ETC_SKETCH_EXHAUSTIVE) {
    if (P > 8) return ETC_ERR_WORKSPACE;
    sketch_exhaustive_kernel<<<1, SK_THREADS, 0, st>>>(d_overlap, n_new, P, d_avail, d_device_map, d_local_bytes);
  } else if (method == ETC_SKETCH_HUNGARIAN) {
    if (P > ETC_SKETCH_MAX_P) return ETC_ERR_WORKSPACE;
    if (P <= 32) {
      sketch_hungarian_warp_kernel<<<1, 32, 0, st>>>(d_overlap, n_new, P, d_avail, d_device_map, d_local_bytes);
      ETC_CUDA_TRY(cudaGetLastError());
      count_launch();
      return ETC_OK;
    }
    // the row-maximum certificate first (a few microseconds); the search below leaves at once if it succeeded
    const int after_tight = P <= TIGHT_MAX ? 1 : 0;
    if (after_tight) {
      char* ws = nullptr;                                       // rowmax [N] | cnt [N] | tight [N][TK]
      const size_t o_cnt = sizeof(int64_t) * (size_t)n_new, o_tight = o_cnt + sizeof(int32_t) * (size_t)n_new;
      ETC_CUDA_TRY(cudaMallocAsync(&ws, o_tight + sizeof(int32_t) * (size_t)n_new * TK, st));
      int64_t* rowmax = reinterpret_cast<int64_t*>(ws);
      int32_t* cnt = reinterpret_cast<int32_t*>(ws + o_cnt); int32_t* tight = reinterpret_cast<int32_t*>(ws + o_tight);
      sketch_rowmax_kernel<<<(n_new + RM_WARPS - 1) / RM_WARPS, RM_WARPS * 32, 0, st>>>(d_overlap, n_new, P, d_avail, rowmax, cnt, tight);
      sketch_tight_kernel<<<1, SK_THREADS, 0, st>>>(n_new, P, d_avail, rowmax, cnt, tight, d_device_map, d_local_bytes);
      const cudaError_t le = cudaGetLastError();
      cudaFreeAsync(ws, st);
      ETC_CUDA_TRY(le);
      count_launch(2);
    }
    const size_t smem = (size_t)n_new * 8 + (size_t)P * 8;       // <= 32 KB: below the default dynamic limit
#define SK_LAUNCH(T, CPT) sketch_hungarian_kernel<T, CPT><<<1, T, smem, st>>>(d_overlap, n_new, P, d_avail, d_device_map, d_local_bytes, after_tight)
    if (P <= 64) SK_LAUNCH(64, 1);
    else if (P <= 128) SK_LAUNCH(128, 1);
    else if (P <= 256) SK_LAUNCH(256, 1);
    else if (P <= 512) SK_LAUNCH(512, 1);
    else if (P <= 1024) SK_LAUNCH(1024, 1);
    else SK_LAUNCH(1024, 2);
#undef SK_LAUNCH
  } else {
    return ETC_ERR_INVALID_ARG;
  }
  ETC_CUDA_TRY(cudaGetLastError());
  count_launch();
  return ETC_OK;
}

// ---------------------------------------------------------------------------------------------- etc_sketch_static
// The sketch for callers that must not allocate (include/etc.h has the user-facing text).  etc_sketch above takes the
// work area of the row-maximum certificate (rowmax [N] int64 | cnt [N] int32 | tight [N][TK] int32) from the
// stream-ordered pool on every call with P > 32; here the same three arrays live in ONE array that is part of the
// library's device image, sized for the largest matrix the certificate handles (TIGHT_MAX rows: 28 KB).  Every GPU that
// loads libetc.so carries those 28 KB from the moment the module is loaded until the process exits.
namespace etc {

constexpr size_t STATIC_SCRATCH_BYTES = (size_t)TIGHT_MAX * (sizeof(int64_t) + sizeof(int32_t) + sizeof(int32_t) * TK);
static_assert(STATIC_SCRATCH_BYTES == ETC_SKETCH_STATIC_SCRATCH_BYTES, "etc.h states the size of the resident work area");
static_assert(TIGHT_MAX == ETC_SKETCH_STATIC_MAX_P, "etc.h states the largest P of etc_sketch_static");
static __device__ __align__(256) unsigned char g_sketch_static_scratch[STATIC_SCRATCH_BYTES];

// In host code `g_sketch_static_scratch` is only a handle for the runtime: it is NOT the array's address on the GPU, and a
// kernel handed it would read and write somewhere else.  The address on a given GPU comes from cudaGetSymbolAddress, asked
// once per device while that device is current, and is remembered here.
constexpr int STATIC_MAX_DEVICES = 64;
static std::mutex g_static_mu;
static unsigned char* g_static_addr[STATIC_MAX_DEVICES] = {};

static cudaError_t sketch_static_scratch(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_sketch_static_scratch);      // no allocation: the array came with the module
    if (e != cudaSuccess) return e;
    g_static_addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_static_addr[dev];
  return cudaSuccess;
}

}  // namespace etc

extern "C" etc_status etc_sketch_static(const int64_t* d_overlap, int32_t n_new, int32_t P, const uint8_t* d_avail,
                                        int32_t* d_device_map, int64_t* d_local_bytes, void* stream) {
  clear_error_detail();
  if (!d_overlap || !d_device_map || !d_local_bytes || n_new < 1 || P < n_new) return ETC_ERR_INVALID_ARG;
  if (P > ETC_SKETCH_STATIC_MAX_P) {
    char msg[160];
    snprintf(msg, sizeof msg, "etc_sketch_static: P = %d exceeds ETC_SKETCH_STATIC_MAX_P = %d (the resident work area holds "
             "%d rows); use etc_sketch", (int)P, (int)ETC_SKETCH_STATIC_MAX_P, (int)ETC_SKETCH_STATIC_MAX_P);
    etc::set_error_text(msg);
    return ETC_ERR_WORKSPACE;
  }
  etc::DeviceGuard device_guard;                 // the library's device is current from here on (the address is per device)
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  cudaStream_t st = (cudaStream_t)stream;
  if (P <= 32) {                                 // one warp, everything on chip: never needed a work area
    sketch_hungarian_warp_kernel<<<1, 32, 0, st>>>(d_overlap, n_new, P, d_avail, d_device_map, d_local_bytes);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
    return ETC_OK;
  }
  unsigned char* ws = nullptr;
  ETC_CUDA_TRY(sketch_static_scratch(&ws));
  // Same carving as etc_sketch.  Nothing in the work area has to start at zero: sketch_rowmax_kernel writes rowmax[n] and
  // cnt[n] for every row before sketch_tight_kernel reads them, and of tight[n][*] only the first cnt[n] entries — written
  // in this call — are ever used; what an earlier call left behind the valid entries is loaded and ignored.
  const size_t o_cnt = sizeof(int64_t) * (size_t)n_new, o_tight = o_cnt + sizeof(int32_t) * (size_t)n_new;
  int64_t* rowmax = reinterpret_cast<int64_t*>(ws);
  int32_t* cnt = reinterpret_cast<int32_t*>(ws + o_cnt); int32_t* tight = reinterpret_cast<int32_t*>(ws + o_tight);
  sketch_rowmax_kernel<<<(n_new + RM_WARPS - 1) / RM_WARPS, RM_WARPS * 32, 0, st>>>(d_overlap, n_new, P, d_avail, rowmax, cnt, tight);
  sketch_tight_kernel<<<1, SK_THREADS, 0, st>>>(n_new, P, d_avail, rowmax, cnt, tight, d_device_map, d_local_bytes);
  ETC_CUDA_TRY(cudaGetLastError());
  const size_t smem = (size_t)n_new * 8 + (size_t)P * 8;         // <= 16 KB
#define SK_LAUNCH(T) sketch_hungarian_kernel<T, 1><<<1, T, smem, st>>>(d_overlap, n_new, P, d_avail, d_device_map, d_local_bytes, 1)
  if (P <= 64) SK_LAUNCH(64);
  else if (P <= 128) SK_LAUNCH(128);
  else if (P <= 256) SK_LAUNCH(256);
  else if (P <= 512) SK_LAUNCH(512);
  else SK_LAUNCH(1024);
#undef SK_LAUNCH
  ETC_CUDA_TRY(cudaGetLastError());
  count_launch(3);
  return ETC_OK;
}
