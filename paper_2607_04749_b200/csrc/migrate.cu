// migrate.cu — (a5) pack, (a6) unpack + local: the HBM-bound hot loop ("The states can be packed to the
// instructions when Send and then unpacked to update the corresponding state after migration"; :195 Refer).
//
// Pure byte movement: a batched gather/scatter over the plan's chunk list.  One CTA copies one chunk (<= 64 KB):
// nrows x row_bytes with independent row pitches on the two sides, through 16-byte streaming loads/stores, four
// independent vectors in flight per thread.  Chunks whose addresses are not 16-byte aligned fall back to the widest
// aligned access (8/4/2/1 bytes).  Two launches per migration:
//   launch 1: pack (old buffers -> staging segments)  +  local slices (old buffer -> new buffer directly)
//   launch 2: unpack (staging segments -> new buffers)
#include <vector>
#include "etc_internal.h"
#include "plan_types.h"

namespace etc {

constexpr int CP_THREADS = 256;
constexpr int CP_UNROLL = 4;

template <typename V> __device__ __forceinline__ V ld_stream(const V* p) { return __ldcs(p); }
template <typename V> __device__ __forceinline__ void st_stream(V* p, const V& v) { __stcs(p, v); }

// copy nrows x row_bytes; V = access type, all addresses and row_bytes are multiples of sizeof(V)
template <typename V>
__device__ __forceinline__ void copy_chunk(const char* __restrict__ src, char* __restrict__ dst, int nrows,
                                           uint32_t row_bytes, uint32_t src_pitch, uint32_t dst_pitch) {
  const uint32_t vpr = row_bytes / (uint32_t)sizeof(V);          // vectors per row
  const uint32_t total = vpr * (uint32_t)nrows;
  const uint32_t tid = threadIdx.x;
  if (nrows == 1) {
    const V* s = reinterpret_cast<const V*>(src); V* d = reinterpret_cast<V*>(dst);
    uint32_t i = tid;
    for (; i + (CP_UNROLL - 1) * CP_THREADS < total; i += CP_UNROLL * CP_THREADS) {
      V v[CP_UNROLL];
#pragma unroll
      for (int k = 0; k < CP_UNROLL; ++k) v[k] = ld_stream(s + i + k * CP_THREADS);
#pragma unroll
      for (int k = 0; k < CP_UNROLL; ++k) st_stream(d + i + k * CP_THREADS, v[k]);
    }
    for (; i < total; i += CP_THREADS) st_stream(d + i, ld_stream(s + i));
    return;
  }
  // 2-D: vector index -> (row, col) with a multiply-high reciprocal (exact for total*vpr < 2^32; here <= 2^32/16)
  const uint32_t magic = (uint32_t)((0x100000000ull + vpr - 1) / vpr);
  auto addr = [&](uint32_t v, const V*& s, V*& d) {
    const uint32_t row = vpr == 1 ? v : __umulhi(v, magic), col = v - row * vpr;
    s = reinterpret_cast<const V*>(src + (size_t)row * src_pitch) + col;
    d = reinterpret_cast<V*>(dst + (size_t)row * dst_pitch) + col;
  };
  uint32_t i = tid;
  for (; i + (CP_UNROLL - 1) * CP_THREADS < total; i += CP_UNROLL * CP_THREADS) {
    V v[CP_UNROLL]; V* d[CP_UNROLL];
#pragma unroll
    for (int k = 0; k < CP_UNROLL; ++k) { const V* s; addr(i + k * CP_THREADS, s, d[k]); v[k] = ld_stream(s); }
#pragma unroll
    for (int k = 0; k < CP_UNROLL; ++k) st_stream(d[k], v[k]);
  }
  for (; i < total; i += CP_THREADS) { const V* s; V* d; addr(i, s, d); st_stream(d, ld_stream(s)); }
}

__device__ __forceinline__ void copy_dispatch(int vec, const char* src, char* dst, int nrows, uint32_t row_bytes,
                                              uint32_t sp, uint32_t dp) {
  switch (vec) {
    case 16: copy_chunk<uint4>(src, dst, nrows, row_bytes, sp, dp); break;
    case 8: copy_chunk<uint2>(src, dst, nrows, row_bytes, sp, dp); break;
    case 4: copy_chunk<unsigned int>(src, dst, nrows, row_bytes, sp, dp); break;
    case 2: copy_chunk<unsigned short>(src, dst, nrows, row_bytes, sp, dp); break;
    default: copy_chunk<unsigned char>(src, dst, nrows, row_bytes, sp, dp); break;
  }
}

// UNPACK = false: blocks [0,nA) pack staged chunks (src -> staging), blocks [nA,nA+nB) copy local chunks (src -> dst)
// UNPACK = true : blocks [0,nA) unpack staged chunks (staging -> dst)
template <bool UNPACK>
__global__ void __launch_bounds__(CP_THREADS)
migrate_copy_kernel(const Chunk* __restrict__ chA, long long nA, const Chunk* __restrict__ chB,
                    const void* const* __restrict__ src_tab, void* const* __restrict__ dst_tab,
                    char* __restrict__ staging) {
  const long long b = blockIdx.x;
  const bool staged = b < nA;
  const Chunk c = staged ? chA[b] : chB[b - nA];
  const char* src; char* dst; uint32_t sp, dp;
  if (UNPACK) {
    src = staging + c.stg_off; sp = (uint32_t)c.row_bytes;
    dst = static_cast<char*>(dst_tab[c.dst_buf]) + c.dst_off; dp = (uint32_t)c.dst_stride;
  } else if (staged) {
    src = static_cast<const char*>(src_tab[c.src_buf]) + c.src_off; sp = (uint32_t)c.src_stride;
    dst = staging + c.stg_off; dp = (uint32_t)c.row_bytes;
  } else {
    src = static_cast<const char*>(src_tab[c.src_buf]) + c.src_off; sp = (uint32_t)c.src_stride;
    dst = static_cast<char*>(dst_tab[c.dst_buf]) + c.dst_off; dp = (uint32_t)c.dst_stride;
  }
  copy_dispatch(c.vec, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp);
}

}  // namespace etc

using namespace etc;

// Validate the caller's pointer tables (only the buffers of `only_kind` if >= 0: the other kinds may already be
// released or not yet allocated), upload them into `d_ptrs`, and launch the copy kernels over the given
// chunk ranges.  `staging` is addressed relative to stg_base.
static etc_status launch_migrate(const etc_plan* pl, const void* const* src_bufs, void* const* dst_bufs, void* staging,
                                 int32_t phases, cudaStream_t st, void** d_ptrs, int only_kind, long long ca, long long nA,
                                 long long la, long long nB, int64_t stg_base, int64_t stg_need) {
  if (!pl || !src_bufs || !dst_bufs || phases < 1 || phases > ETC_PHASE_ALL) return ETC_ERR_INVALID_ARG;
  if (stg_need > 0 && !staging) return ETC_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(staging) & 15) return ETC_ERR_INVALID_ARG;
  const size_t ns = (size_t)pl->n_old * ETC_NUM_KINDS, nd = (size_t)pl->n_new * ETC_NUM_KINDS;
  for (size_t i = 0; i < ns; ++i) {
    if (only_kind >= 0 && (int)(i % ETC_NUM_KINDS) != only_kind) continue;
    if (pl->old_bytes[i] > 0 && !src_bufs[i]) return ETC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(src_bufs[i]) & 15) return ETC_ERR_INVALID_ARG;
  }
  for (size_t i = 0; i < nd; ++i) {
    if (only_kind >= 0 && (int)(i % ETC_NUM_KINDS) != only_kind) continue;
    if (pl->new_bytes[i] > 0 && !dst_bufs[i]) return ETC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(dst_bufs[i]) & 15) return ETC_ERR_INVALID_ARG;
  }
  pl->streams.note(st);
  // pointer tables: source pointers then destination pointers
  ETC_CUDA_TRY(cudaMemcpyAsync(d_ptrs, src_bufs, sizeof(void*) * ns, cudaMemcpyHostToDevice, st));
  ETC_CUDA_TRY(cudaMemcpyAsync(d_ptrs + ns, dst_bufs, sizeof(void*) * nd, cudaMemcpyHostToDevice, st));
  const void* const* d_src = d_ptrs; void* const* d_dst = d_ptrs + ns;
  char* stg = static_cast<char*>(staging) - stg_base;          // chunk records carry offsets of the full staging layout
  if ((phases & ETC_PHASE_PACK) && nA + nB > 0) {
    migrate_copy_kernel<false><<<(unsigned)(nA + nB), CP_THREADS, 0, st>>>(pl->d_ch_staged + ca, nA, pl->d_ch_local + la,
                                                                           d_src, d_dst, stg);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
  }
  if ((phases & ETC_PHASE_UNPACK) && nA > 0) {
    migrate_copy_kernel<true><<<(unsigned)nA, CP_THREADS, 0, st>>>(pl->d_ch_staged + ca, nA, nullptr, d_src, d_dst, stg);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
  }
  return ETC_OK;
}

extern "C" etc_status etc_migrate_phase(const etc_plan* pl, const void* const* src_bufs, void* const* dst_bufs,
                                        void* staging, int32_t phases, void* stream) {
  clear_error_detail();
  if (!pl) return ETC_ERR_INVALID_ARG;
  const PlanTotals& t = pl->totals;
  return launch_migrate(pl, src_bufs, dst_bufs, staging, phases, (cudaStream_t)stream, pl->d_ptrs, -1, 0,
                        t.n_chunks_staged, 0, t.n_chunks_local, 0, t.staging_bytes);
}

extern "C" etc_status etc_migrate(const etc_plan* pl, const void* const* src_bufs, void* const* dst_bufs, void* staging,
                                  void* stream) {
  return etc_migrate_phase(pl, src_bufs, dst_bufs, staging, ETC_PHASE_ALL, stream);
}

// (f2) one round of state chunking: see rounds.cu
extern "C" etc_status etc_migrate_round(const etc_plan* pl, int32_t round, const void* const* src_bufs,
                                        void* const* dst_bufs, void* staging, int32_t phases, void* stream) {
  clear_error_detail();
  if (!pl || round < 0 || (size_t)round >= pl->rounds.size()) return ETC_ERR_INVALID_ARG;
  const RoundRec& r = pl->rounds[round];
  const size_t n_ptrs = ((size_t)(pl->n_old + pl->n_new) * ETC_NUM_KINDS * sizeof(void*) + 255) / 256 * 256 / sizeof(void*);
  return launch_migrate(pl, src_bufs, dst_bufs, staging, phases, (cudaStream_t)stream,
                        pl->d_round_ptrs + n_ptrs * (size_t)round, r.kind, r.ca, r.cb - r.ca, r.la, r.lb - r.la,
                        r.stg_base, r.stg_span);
}
