// plan_order.cu — address-ordered launch lists for the copy kernels (part of (a4); serves (a5)/(a6)).
//
// plan_fill_kernel emits the copy work items ("chunks") unit by unit, a unit being one (source device, new rank) cell of
// the traffic matrix.  Launched in that order, CTAs that run at the same time work on one unit, and two things are lost:
//   * a TP change cuts row-parallel weights into column blocks, so the chunks of DIFFERENT new ranks read interleaved
//     pieces of the same source rows (pack: 64-byte rows out of a 128 ... 512-byte pitch).  Far apart in time, each of
//     them opens every DRAM page of the region for a fraction of its bytes: measured 4.6 TB/s for 64-byte rows and
//     2.9 TB/s for 32-byte rows against 6.8 / 6.2 TB/s when the chunks sharing the rows run side by side;
//   * a source range that several new ranks need (replicated bf16 parameters fanning out to more DP groups, c4) is read
//     from DRAM once per reader, although readers that run together would share it in the 126 MB L2.
// So the plan keeps a second copy of the chunk records in the order the launches should walk them: launch 1 (pack +
// local) sorted by SOURCE address, launch 2 (unpack) sorted by DESTINATION address — in both the side that can be
// strided or shared; the staging side is dense and read / written exactly once either way.  The records are copied, not
// indexed: an index array would put a dependent load in front of every CTA's first access.
//
// The sort is a counting sort over address bins of >= 64 KB of the concatenated buffers (one atomic per chunk for the
// histogram and the rank inside the bin, a two-level exclusive scan of the bins, one scatter); the order inside a bin —
// chunks of one bin touch the same 64 KB, so it does not matter for speed — is then fixed by a per-bin insertion sort,
// so that the lists are deterministic.
#include <algorithm>
#include <vector>
#include "etc_internal.h"
#include "plan_types.h"

namespace etc {

constexpr int ORD_THREADS = 256;
constexpr int SCAN_TILE = 4096;                       // bins per CTA of the two scan kernels (1024 threads x 4)

__device__ __forceinline__ uint32_t bin_of(const int64_t* __restrict__ base, int buf, int64_t off, int shift) {
  return (uint32_t)((base[buf] + off) >> shift);
}

// one thread per chunk: histogram of the address bins; the value the atomic returns is the chunk's rank inside its bin
__global__ void __launch_bounds__(ORD_THREADS)
order_hist_kernel(const Chunk* __restrict__ chA, long long nA, const Chunk* __restrict__ chB, long long nB,
                  const int64_t* __restrict__ obase, const int64_t* __restrict__ nbase, int shift1, int shift2,
                  uint32_t* __restrict__ bins1, uint32_t* __restrict__ bins2, uint32_t* __restrict__ rank1,
                  uint32_t* __restrict__ rank2, const PlanTotals* __restrict__ lazy) {
  const long long i = (long long)blockIdx.x * ORD_THREADS + threadIdx.x;
  if (lazy) { nA = lazy->n_chunks_staged; nB = lazy->n_chunks_local; }   // ETC_NO_SYNC: the grid is an upper bound
  if (i >= nA + nB) return;
  const Chunk* c = i < nA ? chA + i : chB + (i - nA);
  const int sb = c->src_buf; const int64_t so = c->src_off;
  rank1[i] = atomicAdd(&bins1[bin_of(obase, sb, so, shift1)], 1u);
  if (i < nA) rank2[i] = atomicAdd(&bins2[bin_of(nbase, c->dst_buf, c->dst_off, shift2)], 1u);
}

__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* s_w, uint32_t& total) {   // 1024 threads
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  if (lane == 31) s_w[wid] = x;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = s_w[lane], z = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, z, o); if (lane >= o) z += y; }
    s_w[lane] = z - w;                                 // exclusive prefix of the warp totals
    if (lane == 31) s_w[32] = z;                       // block total
  }
  __syncthreads();
  total = s_w[32];
  const uint32_t r = s_w[wid] + x - v;
  __syncthreads();
  return r;
}

// scan level 1: sum of each tile of SCAN_TILE bins
__global__ void __launch_bounds__(1024) order_tile_sums_kernel(const uint32_t* __restrict__ bins, long long n, uint32_t* __restrict__ sums) {
  __shared__ uint32_t s_w[33];
  const long long i0 = (long long)blockIdx.x * SCAN_TILE + threadIdx.x * 4;
  uint32_t v = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) if (i0 + k < n) v += bins[i0 + k];
  uint32_t tot; block_excl_scan(v, s_w, tot);
  if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

// scan level 2: every CTA adds up the tiles before its own (<= a few thousand values) and scans its tile in place
__global__ void __launch_bounds__(1024) order_scan_kernel(uint32_t* __restrict__ bins, long long n, const uint32_t* __restrict__ sums) {
  __shared__ uint32_t s_w[33];
  uint32_t pre = 0;
  for (int t = threadIdx.x; t < (int)blockIdx.x; t += 1024) pre += sums[t];
  uint32_t base; block_excl_scan(pre, s_w, base);      // base = sum of all earlier tiles
  const long long i0 = (long long)blockIdx.x * SCAN_TILE + threadIdx.x * 4;
  uint32_t b[4], v = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) { b[k] = i0 + k < n ? bins[i0 + k] : 0; v += b[k]; }
  uint32_t tot; uint32_t ex = base + block_excl_scan(v, s_w, tot);
#pragma unroll
  for (int k = 0; k < 4; ++k) { if (i0 + k < n) bins[i0 + k] = ex; ex += b[k]; }
}

// one thread per chunk: the record goes to (first position of its bin) + (its rank inside the bin).  bins2 continues the
// scan of bins1, whose total is nA + nB.
__global__ void __launch_bounds__(ORD_THREADS)
order_scatter_kernel(const Chunk* __restrict__ chA, long long nA, const Chunk* __restrict__ chB, long long nB,
                     const int64_t* __restrict__ obase, const int64_t* __restrict__ nbase, int shift1, int shift2,
                     const uint32_t* __restrict__ bins1, const uint32_t* __restrict__ bins2,
                     const uint32_t* __restrict__ rank1, const uint32_t* __restrict__ rank2, Chunk* __restrict__ out1,
                     Chunk* __restrict__ out2, const PlanTotals* __restrict__ lazy) {
  const long long i = (long long)blockIdx.x * ORD_THREADS + threadIdx.x;
  if (lazy) { nA = lazy->n_chunks_staged; nB = lazy->n_chunks_local; }
  if (i >= nA + nB) return;
  Chunk c = i < nA ? chA[i] : chB[i - nA];
  if (i < nA) out2[bins2[bin_of(nbase, c.dst_buf, c.dst_off, shift2)] - (uint32_t)(nA + nB) + rank2[i]] = c;
  c.pad = i < nA ? CHUNK_STAGED : 0;                   // list 1 mixes staged and local chunks
  out1[bins1[bin_of(obase, c.src_buf, c.src_off, shift1)] + rank1[i]] = c;
}

// The atomics above leave the order INSIDE a bin to chance.  One thread per bin puts its few records (typically 1-8: a bin is
// 64 KB of one buffer) into a fixed order — list 1 by (source offset, destination buffer, destination offset), list 2 by
// (destination offset, source buffer, source offset) — so that a plan's launch lists are the same on every run.
__device__ __forceinline__ bool rec_less(const Chunk& a, const Chunk& b, bool by_src) {
  if (by_src) {
    if (a.src_off != b.src_off) return a.src_off < b.src_off;
    if (a.dst_buf != b.dst_buf) return a.dst_buf < b.dst_buf;
    if (a.dst_off != b.dst_off) return a.dst_off < b.dst_off;
    return a.stg_off < b.stg_off;
  }
  if (a.dst_off != b.dst_off) return a.dst_off < b.dst_off;
  if (a.src_buf != b.src_buf) return a.src_buf < b.src_buf;
  return a.src_off < b.src_off;
}
__global__ void __launch_bounds__(ORD_THREADS)
order_bin_sort_kernel(const uint32_t* __restrict__ bins, long long n1, long long n2, long long nA, long long nB,
                      Chunk* __restrict__ out1, Chunk* __restrict__ out2, const PlanTotals* __restrict__ lazy) {
  const long long b = (long long)blockIdx.x * ORD_THREADS + threadIdx.x;
  if (b >= n1 + n2) return;
  if (lazy) { nA = lazy->n_chunks_staged; nB = lazy->n_chunks_local; }
  const bool first = b < n1;
  const uint32_t total = (uint32_t)(first ? nA + nB : nA + nB + nA);        // the scan runs on through both bin tables
  const uint32_t lo = bins[b], hi = (b + 1 == n1 + n2) ? total : (b + 1 == n1 ? (uint32_t)(nA + nB) : bins[b + 1]);
  if (hi <= lo + 1) return;
  Chunk* r = first ? out1 + lo : out2 + (lo - (uint32_t)(nA + nB));
  const uint32_t n = hi - lo;
  if (n <= 32) {                                                           // insertion sort: the runs are short
    for (uint32_t i = 1; i < n; ++i) {
      const Chunk x = r[i];
      uint32_t j = i;
      while (j > 0 && rec_less(x, r[j - 1], first)) { r[j] = r[j - 1]; --j; }
      if (j != i) r[j] = x;
    }
    return;
  }
  // a crowded bin (many tiny tensors in one 64 KB, or the coarser bins of a very large layout): heap sort, O(n log n)
  auto sift = [&](uint32_t root, uint32_t end) {
    const Chunk x = r[root];
    while (true) {
      uint32_t child = 2 * root + 1;
      if (child >= end) break;
      if (child + 1 < end && rec_less(r[child], r[child + 1], first)) ++child;
      if (!rec_less(x, r[child], first)) break;
      r[root] = r[child]; root = child;
    }
    r[root] = x;
  };
  for (uint32_t i = n / 2; i-- > 0;) sift(i, n);
  for (uint32_t e = n - 1; e > 0; --e) { const Chunk t = r[0]; r[0] = r[e]; r[e] = t; sift(0, e); }
}

// exclusive prefix sums of the buffer sizes, each buffer starting on a bin boundary; returns the number of bins
static long long bases_of(const std::vector<int64_t>& bytes, int shift, std::vector<int64_t>& base) {
  base.resize(bytes.size());
  int64_t run = 0;
  for (size_t i = 0; i < bytes.size(); ++i) { base[i] = run; run += ((bytes[i] >> shift) + 1) << shift; }
  return (long long)(run >> shift) + 1;
}
static int pick_shift(const std::vector<int64_t>& bytes, std::vector<int64_t>& base, long long& n_bins) {
  int shift = 16;                                      // one chunk of payload
  while ((n_bins = bases_of(bytes, shift, base)) > (1ll << 22)) ++shift;
  return shift;
}

// Scratch of the sort, sized for the largest range it will be run on, and the two base tables.
struct OrderScratch {
  char* tmp = nullptr;
  int64_t* d_ob = nullptr; int64_t* d_nb = nullptr;
  uint32_t* bins = nullptr; uint32_t* sums = nullptr; uint32_t* r1 = nullptr; uint32_t* r2 = nullptr;
  int shift1 = 16, shift2 = 16;
  long long n1 = 0, n2 = 0;
};
static cudaError_t scratch_make(const etc_plan* pl, long long max_a, long long max_ab, cudaStream_t st, OrderScratch& s) {
  std::vector<int64_t> ob, nb;
  s.shift1 = pick_shift(pl->old_bytes, ob, s.n1); s.shift2 = pick_shift(pl->new_bytes, nb, s.n2);
  const long long n_bins = s.n1 + s.n2, n_tiles = (n_bins + SCAN_TILE - 1) / SCAN_TILE;
  auto al = [](size_t x) { return (x + 255) & ~size_t(255); };
  const size_t o_ob = 0, o_nb = o_ob + sizeof(int64_t) * ob.size(), o_bins = al(o_nb + sizeof(int64_t) * nb.size()),
               o_sums = o_bins + al(sizeof(uint32_t) * (size_t)n_bins), o_r1 = o_sums + al(sizeof(uint32_t) * (size_t)n_tiles),
               o_r2 = o_r1 + al(sizeof(uint32_t) * (size_t)max_ab), bytes = o_r2 + al(sizeof(uint32_t) * (size_t)max_a);
  cudaError_t e = cudaMallocAsync(&s.tmp, bytes, st);
  if (e != cudaSuccess) return e;
  s.d_ob = reinterpret_cast<int64_t*>(s.tmp + o_ob); s.d_nb = reinterpret_cast<int64_t*>(s.tmp + o_nb);
  s.bins = reinterpret_cast<uint32_t*>(s.tmp + o_bins); s.sums = reinterpret_cast<uint32_t*>(s.tmp + o_sums);
  s.r1 = reinterpret_cast<uint32_t*>(s.tmp + o_r1); s.r2 = reinterpret_cast<uint32_t*>(s.tmp + o_r2);
  ob.insert(ob.end(), nb.begin(), nb.end());                     // both base tables in one upload
  return write_small(s.d_ob, ob.data(), sizeof(int64_t) * ob.size(), st);
}

// Sort one range: staged chunks chA[0,nA), local chunks chB[0,nB) -> out1[0,nA+nB) by source address, out2[0,nA) by
// destination address.
static cudaError_t order_range(const OrderScratch& s, const Chunk* chA, long long nA, const Chunk* chB, long long nB,
                               Chunk* out1, Chunk* out2, cudaStream_t st, const PlanTotals* lazy = nullptr,
                               long long bound = 0) {
  if (!lazy && nA + nB == 0) return cudaSuccess;
  const long long n_bins = s.n1 + s.n2, n_tiles = (n_bins + SCAN_TILE - 1) / SCAN_TILE;
  cudaError_t e = cudaMemsetAsync(s.bins, 0, sizeof(uint32_t) * (size_t)n_bins, st);
  if (e != cudaSuccess) return e;
  const unsigned grid = (unsigned)(((lazy ? bound : nA + nB) + ORD_THREADS - 1) / ORD_THREADS);
  order_hist_kernel<<<grid, ORD_THREADS, 0, st>>>(chA, nA, chB, nB, s.d_ob, s.d_nb, s.shift1, s.shift2, s.bins, s.bins + s.n1,
                                                   s.r1, s.r2, lazy);
  order_tile_sums_kernel<<<(unsigned)n_tiles, 1024, 0, st>>>(s.bins, n_bins, s.sums);
  order_scan_kernel<<<(unsigned)n_tiles, 1024, 0, st>>>(s.bins, n_bins, s.sums);
  order_scatter_kernel<<<grid, ORD_THREADS, 0, st>>>(chA, nA, chB, nB, s.d_ob, s.d_nb, s.shift1, s.shift2, s.bins, s.bins + s.n1,
                                                      s.r1, s.r2, out1, out2, lazy);
  order_bin_sort_kernel<<<(unsigned)((n_bins + ORD_THREADS - 1) / ORD_THREADS), ORD_THREADS, 0, st>>>(s.bins, s.n1, s.n2, nA, nB,
                                                                                                    out1, out2, lazy);
  count_launch(5);
  return cudaGetLastError();
}

static size_t list_bytes(long long n) { return ((sizeof(Chunk) * (size_t)n) + 255) & ~size_t(255); }

// Build pl->d_ch1 / pl->d_ch2 from the finished chunk lists on `st`.  nA, nB: the chunk counts — or, for an ETC_NO_SYNC
// plan (`lazy` = its device-side totals), the bound both lists together stay below: grids and lists are then sized by
// the bound and the kernels read the counts from `lazy`.
cudaError_t plan_build_order(etc_plan* pl, long long nA, long long nB, cudaStream_t st, const PlanTotals* lazy) {
  if (lazy) nA = nB = std::max(nA, nB);
  if (nA + nB == 0 || nA + nB >= (1ll << 32)) return cudaSuccess;
  const long long n1 = lazy ? nA : nA + nB;                      // capacity of list 1
  cudaError_t e = cudaMallocAsync(&pl->d_order_ws, list_bytes(n1) + list_bytes(nA), st);
  if (e != cudaSuccess) return e;
  Chunk* out1 = static_cast<Chunk*>(pl->d_order_ws);
  Chunk* out2 = reinterpret_cast<Chunk*>(static_cast<char*>(pl->d_order_ws) + list_bytes(n1));
  OrderScratch s;
  e = scratch_make(pl, nA, n1, st, s);
  if (e == cudaSuccess) e = order_range(s, pl->d_ch_staged, nA, pl->d_ch_local, nB, out1, out2, st, lazy, n1);
  if (s.tmp) cudaFreeAsync(s.tmp, st);
  if (e == cudaSuccess) { pl->d_ch1 = out1; pl->d_ch2 = out2; }
  return e;
}

// The same per round of state chunking (rounds.cu): round i covers staged chunks [ca,cb) and local chunks [la,lb); its
// ordered launch-1 list is d_rch1[ca + la, cb + lb), its launch-2 list d_rch2[ca, cb).
cudaError_t plan_build_round_order(etc_plan* pl, cudaStream_t st) {
  if (!pl->d_ch1 || pl->rounds.empty()) return cudaSuccess;      // the plan launches in list order
  const PlanTotals& t = plan_totals(pl);
  const long long nA = t.n_chunks_staged, nB = t.n_chunks_local;
  long long max_a = 0, max_ab = 0;
  for (const RoundRec& r : pl->rounds) { max_a = std::max<long long>(max_a, r.cb - r.ca); max_ab = std::max<long long>(max_ab, r.cb - r.ca + r.lb - r.la); }
  if (max_ab == 0) return cudaSuccess;
  cudaError_t e = cudaMallocAsync(&pl->d_round_order_ws, list_bytes(nA + nB) + list_bytes(nA), st);
  if (e != cudaSuccess) return e;
  Chunk* out1 = static_cast<Chunk*>(pl->d_round_order_ws);
  Chunk* out2 = reinterpret_cast<Chunk*>(static_cast<char*>(pl->d_round_order_ws) + list_bytes(nA + nB));
  OrderScratch s;
  e = scratch_make(pl, max_a, max_ab, st, s);
  for (size_t i = 0; e == cudaSuccess && i < pl->rounds.size(); ++i) {
    const RoundRec& r = pl->rounds[i];
    e = order_range(s, pl->d_ch_staged + r.ca, r.cb - r.ca, pl->d_ch_local + r.la, r.lb - r.la, out1 + r.ca + r.la, out2 + r.ca, st);
  }
  if (s.tmp) cudaFreeAsync(s.tmp, st);
  if (e == cudaSuccess) { pl->d_rch1 = out1; pl->d_rch2 = out2; }
  return e;
}

}  // namespace etc
