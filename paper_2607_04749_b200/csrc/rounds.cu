// rounds.cu — (f2) state chunking with bounded staging and eager release ("we use state chunking to migrate
// states in sequential chunks with on-demand buffer allocation, and eager release of source-side state to promptly free
// source-side tensors after each round"; :378 "ETC reduces the peak to one optimizer component at a time").
//
// A kind-major plan (ETC_KIND_MAJOR) orders units, slices, chunks and staging segments by state kind first, so the work
// of one optimizer component is one contiguous range of every table.  A round = (kind, window j): the staged chunks of
// that kind whose staging offset starts inside window j of `window` bytes, plus the j-th share of the kind's local
// chunks.  A chunk is at most ETC_CHUNK_BYTES long, so a round touches at most window + ETC_CHUNK_BYTES <= the caller's
// bound of staging, addressed relative to the window start.  Rounds of one kind read only that kind's source buffers and
// write only that kind's destination buffers: after the kind's last round the caller may free its source buffers, and
// it need not allocate a kind's destination buffers before the kind's first round.
//
// Window boundaries are found independently per round by binary search over the (monotone) staging offsets of the
// chunk table: one CTA per round, which then reduces the round's payload bytes.
#include <algorithm>
#include <cstring>
#include <vector>
#include "etc_internal.h"
#include "plan_types.h"

namespace etc {

struct RoundSpec { int64_t c_lo, c_hi, stg_lo, stg_hi; int64_t la, lb; };   // search range, window, local share

__device__ __forceinline__ long long lower_bound_stg(const Chunk* ch, long long lo, long long hi, int64_t key) {
  while (lo < hi) { const long long mid = (lo + hi) >> 1; if (ch[mid].stg_off < key) lo = mid + 1; else hi = mid; }
  return lo;
}

__global__ void __launch_bounds__(256)
plan_rounds_kernel(const Chunk* __restrict__ ch_staged, const Chunk* __restrict__ ch_local,
                   const RoundSpec* __restrict__ specs, RoundRec* __restrict__ out) {
  __shared__ long long s_ca, s_cb;
  __shared__ int64_t s_red[2][8];
  const RoundSpec sp = specs[blockIdx.x];
  if (threadIdx.x == 0) s_ca = lower_bound_stg(ch_staged, sp.c_lo, sp.c_hi, sp.stg_lo);
  if (threadIdx.x == 32) s_cb = lower_bound_stg(ch_staged, sp.c_lo, sp.c_hi, sp.stg_hi);
  __syncthreads();
  const long long ca = s_ca, cb = s_cb;
  int64_t sb = 0, lb = 0;
  for (long long i = ca + threadIdx.x; i < cb; i += blockDim.x) sb += (int64_t)ch_staged[i].nrows * ch_staged[i].row_bytes;
  for (long long i = sp.la + threadIdx.x; i < sp.lb; i += blockDim.x) lb += (int64_t)ch_local[i].nrows * ch_local[i].row_bytes;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { sb += __shfl_xor_sync(0xffffffffu, sb, o); lb += __shfl_xor_sync(0xffffffffu, lb, o); }
  if ((threadIdx.x & 31) == 0) { s_red[0][threadIdx.x >> 5] = sb; s_red[1][threadIdx.x >> 5] = lb; }
  __syncthreads();
  if (threadIdx.x == 0) {
    sb = lb = 0;
    for (int w = 0; w < 8; ++w) { sb += s_red[0][w]; lb += s_red[1][w]; }
    RoundRec& r = out[blockIdx.x];
    r.ca = ca; r.cb = cb; r.la = sp.la; r.lb = sp.lb;
    r.stg_base = sp.stg_lo; r.staged_bytes = sb; r.local_bytes = lb;
    r.stg_span = 0;
    if (cb > ca) { const Chunk& last = ch_staged[cb - 1]; r.stg_span = last.stg_off + (int64_t)last.nrows * last.row_bytes - sp.stg_lo; }
  }
}

}  // namespace etc

using namespace etc;

extern "C" etc_status etc_plan_set_rounds(etc_plan* pl, int64_t max_staging_bytes, int32_t* n_rounds, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !n_rounds) return ETC_ERR_INVALID_ARG;
  if (!(pl->flags & ETC_KIND_MAJOR)) return ETC_ERR_INVALID_ARG;
  if (max_staging_bytes < 2 * (int64_t)ETC_CHUNK_BYTES) return ETC_ERR_INVALID_ARG;
  const int64_t window = (max_staging_bytes - ETC_CHUNK_BYTES) & ~(int64_t)511;
  cudaStream_t st = (cudaStream_t)stream;
  etc_status plan_rc = ETC_OK;
  const PlanTotals& t = plan_totals(pl, &plan_rc);
  if (plan_rc != ETC_OK) return plan_rc;                       // device-detected error of an ETC_NO_SYNC plan

  std::vector<RoundSpec> specs;
  std::vector<RoundRec> recs;
  for (int k = 0; k < ETC_NUM_KINDS; ++k) {
    const int64_t c_lo = t.kind_base[k][0], c_hi = t.kind_base[k + 1][0];
    const int64_t s_lo = t.kind_base[k][1], s_hi = t.kind_base[k + 1][1];
    const int64_t l_lo = t.kind_base[k][2], l_hi = t.kind_base[k + 1][2];
    if (c_hi == c_lo && l_hi == l_lo) continue;                // the kind moves nothing
    const int64_t J = std::max<int64_t>(1, (s_hi - s_lo + window - 1) / window);
    if ((int64_t)specs.size() + J > (1 << 20)) return ETC_ERR_WORKSPACE;
    for (int64_t j = 0; j < J; ++j) {
      RoundSpec sp;
      sp.c_lo = c_lo; sp.c_hi = c_hi;
      sp.stg_lo = s_lo + j * window; sp.stg_hi = (j + 1 == J) ? INT64_MAX : s_lo + (j + 1) * window;
      const int64_t nl = l_hi - l_lo;                          // local chunks: the j-th of J equal shares
      sp.la = l_lo + (int64_t)((__int128)nl * j / J); sp.lb = l_lo + (int64_t)((__int128)nl * (j + 1) / J);
      specs.push_back(sp);
      RoundRec r{}; r.kind = k; r.sub = (int32_t)j; r.n_sub = (int32_t)J;
      recs.push_back(r);
    }
  }
  const size_t R = specs.size();
  if (pl->d_rounds_ws) { cudaFreeAsync(pl->d_rounds_ws, pl->streams.join(st)); pl->d_rounds_ws = nullptr; pl->d_round_ptrs = nullptr; }
  if (pl->d_round_order_ws) { cudaFreeAsync(pl->d_round_order_ws, pl->streams.join(st)); pl->d_round_order_ws = nullptr; pl->d_rch1 = pl->d_rch2 = nullptr; }
  ETC_CUDA_TRY(plan_use(pl, st));
  pl->rounds.clear(); pl->round_staging_cap = max_staging_bytes;
  *n_rounds = (int32_t)R;
  if (R == 0) return ETC_OK;

  auto al = [](size_t x) { return (x + 255) & ~size_t(255); };
  const size_t n_ptrs = (size_t)(pl->n_old + pl->n_new) * ETC_NUM_KINDS;
  const size_t o_specs = 0, o_recs = al(sizeof(RoundSpec) * R), o_ptrs = o_recs + al(sizeof(RoundRec) * R),
               bytes = o_ptrs + al(sizeof(void*) * n_ptrs) * R;
  ETC_CUDA_TRY(cudaMallocAsync(&pl->d_rounds_ws, bytes, st));
  char* ws = static_cast<char*>(pl->d_rounds_ws);
  pl->d_round_ptrs = reinterpret_cast<void**>(ws + o_ptrs);
  // metadata moves as kernels on `st` while it is small (xfer.cu); a very long round list falls back to DMA copies
  const bool small = R <= 512;
  if (small) ETC_CUDA_TRY(write_small(ws + o_specs, specs.data(), sizeof(RoundSpec) * R, st));
  else ETC_CUDA_TRY(cudaMemcpyAsync(ws + o_specs, specs.data(), sizeof(RoundSpec) * R, cudaMemcpyHostToDevice, st));
  plan_rounds_kernel<<<(unsigned)R, 256, 0, st>>>(pl->d_ch_staged, pl->d_ch_local,
                                                  reinterpret_cast<const RoundSpec*>(ws + o_specs),
                                                  reinterpret_cast<RoundRec*>(ws + o_recs));
  ETC_CUDA_TRY(cudaGetLastError());
  count_launch();
  std::vector<RoundRec> got(R);
  {
    std::lock_guard<std::mutex> lock(pinned_scratch_mutex());
    void* pin = small ? pinned_scratch(sizeof(RoundRec) * R) : nullptr;
    if (pin) ETC_CUDA_TRY(copy_by_kernel(pin, ws + o_recs, sizeof(RoundRec) * R, st));
    else ETC_CUDA_TRY(cudaMemcpyAsync(got.data(), ws + o_recs, sizeof(RoundRec) * R, cudaMemcpyDeviceToHost, st));
    ETC_CUDA_TRY(cudaStreamSynchronize(st));                   // plan-time: round sizes must come back to the host
    if (pin) memcpy(got.data(), pin, sizeof(RoundRec) * R);
  }
  for (size_t i = 0; i < R; ++i) { got[i].kind = recs[i].kind; got[i].sub = recs[i].sub; got[i].n_sub = recs[i].n_sub; }
  pl->rounds = std::move(got);
  ETC_CUDA_TRY(plan_build_round_order(pl, st));                // each round's launch lists in address order (plan_order.cu)
  return ETC_OK;
}

extern "C" etc_status etc_plan_get_round(const etc_plan* pl, int32_t round, etc_round_info* out) {
  if (!pl || !out || round < 0 || (size_t)round >= pl->rounds.size()) return ETC_ERR_INVALID_ARG;
  const RoundRec& r = pl->rounds[round];
  out->kind = r.kind; out->sub = r.sub; out->n_sub = r.n_sub; out->pad = 0;
  out->staging_bytes = r.stg_span; out->staged_bytes = r.staged_bytes; out->local_bytes = r.local_bytes;
  out->n_chunks_staged = r.cb - r.ca; out->n_chunks_local = r.lb - r.la;
  return ETC_OK;
}
