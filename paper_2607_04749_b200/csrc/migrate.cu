// migrate.cu — (a5) pack, (a6) unpack + local: the HBM-bound hot loop ("The states can be packed to the
// instructions when Send and then unpacked to update the corresponding state after migration"; :195 Refer).
//
// Pure byte movement: a batched gather/scatter over the plan's chunk list.  One CTA copies one chunk (<= 64 KB of
// payload): nrows x row_bytes with independent row pitches on the two sides, staged through a 72 KB shared-memory tile
// (three CTAs per SM keep ~192 KB in flight per SM); the hardware block scheduler balances the chunks over the SMs.
// The copy paths (TMA bulk copies, short-row gather / scatter around one bulk copy, byte-phase re-aligning) are in
// copy_paths.cuh.  Two launches per migration:
//   launch 1: pack (old buffers -> staging segments)  +  local slices (old buffer -> new buffer directly)
//   launch 2: unpack (staging segments -> new buffers)
#include <vector>
#include "etc_internal.h"
#include "plan_types.h"
#include "copy_paths.cuh"

namespace etc {

// Pointer tables.  The caller's buffer pointers (n_old*4 source pointers, then n_new*4 destination pointers) ride in the
// kernel's parameter block when they fit (PTR_PARAM_MAX pointers: up to 96 devices in all), so every launch carries its
// own table: concurrent etc_migrate calls on one plan from different streams with different buffer sets (double-
// buffered payloads, a replayed CUDA graph beside a live call) cannot disturb each other, and no upload kernel is
// needed.  Larger device counts use a table in device memory that belongs to the plan (include/etc.h states the
// ordering rule for that case).
constexpr int PTR_PARAM_MAX = 384;
struct PtrParams { const void* p[PTR_PARAM_MAX]; };

// UNPACK = false: blocks [0,nA) pack staged chunks (src -> staging), blocks [nA,nA+nB) copy local chunks (src -> dst)
// UNPACK = true : blocks [0,nA) unpack staged chunks (staging -> dst)
// `ordered` (or null): the same chunks as ONE list in the order the launch should walk them (plan_order.cu: by source
// address for launch 1, staged chunks flagged; by destination address for launch 2); block b then takes ordered[b].
template <bool UNPACK, bool PARAM_PTRS>
__global__ void __launch_bounds__(CP_THREADS)
migrate_copy_kernel(const Chunk* __restrict__ chA, long long nA, const Chunk* __restrict__ chB,
                    const void* const* __restrict__ tab, int ns, char* __restrict__ staging,
                    const PlanTotals* __restrict__ lazy, const Chunk* __restrict__ ordered,
                    const __grid_constant__ PtrParams pp) {
  extern __shared__ __align__(128) char tile[];                 // TILE_BYTES: the staging tile of every copy path
  __shared__ uint64_t bar;
  const long long b = blockIdx.x;
  if (lazy) {                                                   // ETC_NO_SYNC plan: the grid is an upper bound, the counts are here
    nA = lazy->n_chunks_staged;
    if (b >= nA + (UNPACK ? 0 : lazy->n_chunks_local)) return;
  }
  const Chunk c = ordered ? ordered[b] : (b < nA ? chA[b] : chB[b - nA]);
  const bool staged = UNPACK || (ordered ? (c.pad & CHUNK_STAGED) != 0 : b < nA);
  const char* src; char* dst; uint32_t sp, dp;
  auto src_ptr = [&]() { return static_cast<const char*>(PARAM_PTRS ? pp.p[c.src_buf] : tab[c.src_buf]); };
  auto dst_ptr = [&]() { return static_cast<char*>(const_cast<void*>(PARAM_PTRS ? pp.p[ns + c.dst_buf] : tab[ns + c.dst_buf])); };
  if (UNPACK) {
    src = staging + c.stg_off; sp = (uint32_t)c.row_bytes;
    dst = dst_ptr() + c.dst_off; dp = (uint32_t)c.dst_stride;
  } else if (staged) {
    src = src_ptr() + c.src_off; sp = (uint32_t)c.src_stride;
    dst = staging + c.stg_off; dp = (uint32_t)c.row_bytes;
  } else {
    src = src_ptr() + c.src_off; sp = (uint32_t)c.src_stride;
    dst = dst_ptr() + c.dst_off; dp = (uint32_t)c.dst_stride;
  }
  copy_one_chunk(tile, &bar, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp, c.vec);
}

// Zero-fill (reading A31): blockIdx.x = descriptor, blockIdx.y = one of FILL_SPLIT CTAs sharing its rows x row_bytes.
// only_kind >= 0 restricts the launch to one state kind (rounds of state chunking).  Padding rows are a sliver of the
// state, so this is the plain vector store loop, not a tuned kernel.
constexpr int FILL_SPLIT = 16;
template <typename V>
__device__ __forceinline__ void fill_rows(char* dst, int nrows, uint32_t row_bytes, uint32_t pitch) {
  const uint32_t vpr = row_bytes / (uint32_t)sizeof(V);
  const unsigned long long total = (unsigned long long)vpr * (unsigned)nrows;
  V z; memset(&z, 0, sizeof(V));
  for (unsigned long long i = (unsigned long long)blockIdx.y * blockDim.x + threadIdx.x; i < total;
       i += (unsigned long long)gridDim.y * blockDim.x) {
    const unsigned long long row = i / vpr, col = i - row * vpr;
    reinterpret_cast<V*>(dst + row * pitch)[col] = z;
  }
}
template <bool PARAM_PTRS>
__global__ void __launch_bounds__(CP_THREADS)
migrate_fill_kernel(const etc_slice* __restrict__ fills, const void* const* __restrict__ tab, int ns, int only_kind,
                    const PlanTotals* __restrict__ lazy, const __grid_constant__ PtrParams pp) {
  if (lazy && (long long)blockIdx.x >= lazy->n_fills) return;
  const etc_slice f = fills[blockIdx.x];
  if (only_kind >= 0 && f.kind != only_kind) return;
  const int di = ns + f.dst_rank * ETC_NUM_KINDS + f.kind;
  char* dst = static_cast<char*>(const_cast<void*>(PARAM_PTRS ? pp.p[di] : tab[di])) + f.dst_off;
  int64_t al = f.dst_off | f.row_bytes;
  if (f.nrows > 1) al |= (int64_t)f.dst_stride;
  const int64_t low = al & -al;
  // one contiguous run longer than 2^32 bytes cannot occur (a buffer row is < 2^31 elements); rows are < 4 GiB
  if (low >= 16 || al == 0) fill_rows<uint4>(dst, f.nrows, (uint32_t)f.row_bytes, (uint32_t)f.dst_stride);
  else if (low >= 4) fill_rows<unsigned int>(dst, f.nrows, (uint32_t)f.row_bytes, (uint32_t)f.dst_stride);
  else if (low >= 2) fill_rows<unsigned short>(dst, f.nrows, (uint32_t)f.row_bytes, (uint32_t)f.dst_stride);
  else fill_rows<unsigned char>(dst, f.nrows, (uint32_t)f.row_bytes, (uint32_t)f.dst_stride);
}

// the TMA path stages one chunk per CTA in dynamic shared memory; function attributes are per device
template <typename K> static cudaError_t big_smem(K kernel) {
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TILE_BYTES);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  return e;
}
static cudaError_t copy_kernel_attrs() {
  static bool done[64] = {};
  static std::mutex mu;                                         // etc_migrate* may be called from several host threads
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
  e = big_smem(migrate_copy_kernel<false, false>);
  if (e == cudaSuccess) e = big_smem(migrate_copy_kernel<false, true>);
  if (e == cudaSuccess) e = big_smem(migrate_copy_kernel<true, false>);
  if (e == cudaSuccess) e = big_smem(migrate_copy_kernel<true, true>);
  if (e == cudaSuccess && dev >= 0 && dev < 64) done[dev] = true;
  return e;
}

}  // namespace etc

using namespace etc;

// Validate the caller's pointer tables (only the buffers of `only_kind` if >= 0: the other kinds may already be
// released or not yet allocated), upload them into `d_ptrs`, and launch the copy kernels over the given
// chunk ranges.  `staging` is addressed relative to stg_base.
static etc_status launch_migrate(const etc_plan* pl, const void* const* src_bufs, void* const* dst_bufs, void* staging,
                                 int32_t phases, cudaStream_t st, void** d_ptrs, int only_kind, long long ca, long long nA,
                                 long long la, long long nB, int64_t stg_base, int64_t stg_need, bool with_fills,
                                 long long n_fills, const PlanTotals* lazy, const Chunk* order1 = nullptr,
                                 const Chunk* order2 = nullptr) {
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
  ETC_CUDA_TRY(copy_kernel_attrs());
  ETC_CUDA_TRY(plan_use(pl, st));                               // `st` waits for the plan's tables if they were written elsewhere
  // pointer tables: source pointers then destination pointers — in the kernel's parameter block when they fit, else
  // written into the plan's device table by a kernel on `st` (not a DMA copy: it would queue behind bulk transfers)
  const bool in_params = ns + nd <= (size_t)PTR_PARAM_MAX;
  PtrParams pp;
  if (in_params) {
    for (size_t i = 0; i < ns; ++i) pp.p[i] = src_bufs[i];
    for (size_t i = 0; i < nd; ++i) pp.p[ns + i] = dst_bufs[i];
  } else {
    std::vector<const void*> both(ns + nd);
    for (size_t i = 0; i < ns; ++i) both[i] = src_bufs[i];
    for (size_t i = 0; i < nd; ++i) both[ns + i] = dst_bufs[i];
    ETC_CUDA_TRY(write_small(d_ptrs, both.data(), sizeof(void*) * (ns + nd), st));
  }
  const void* const* tab = d_ptrs;
  char* stg = static_cast<char*>(staging) - stg_base;          // chunk records carry offsets of the full staging layout
  if ((phases & ETC_PHASE_PACK) && nA + nB > 0) {
    if (in_params) migrate_copy_kernel<false, true><<<(unsigned)(nA + nB), CP_THREADS, TILE_BYTES, st>>>(
        pl->d_ch_staged + ca, nA, pl->d_ch_local + la, tab, (int)ns, stg, lazy, order1, pp);
    else migrate_copy_kernel<false, false><<<(unsigned)(nA + nB), CP_THREADS, TILE_BYTES, st>>>(
        pl->d_ch_staged + ca, nA, pl->d_ch_local + la, tab, (int)ns, stg, lazy, order1, pp);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
  }
  if ((phases & ETC_PHASE_PACK) && with_fills && n_fills > 0) {                 // reading A31: bytes with no source
    const dim3 grid((unsigned)n_fills, FILL_SPLIT);
    if (in_params) migrate_fill_kernel<true><<<grid, CP_THREADS, 0, st>>>(pl->d_fills, tab, (int)ns, only_kind, lazy, pp);
    else migrate_fill_kernel<false><<<grid, CP_THREADS, 0, st>>>(pl->d_fills, tab, (int)ns, only_kind, lazy, pp);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
  }
  if ((phases & ETC_PHASE_UNPACK) && nA > 0) {
    if (in_params) migrate_copy_kernel<true, true><<<(unsigned)nA, CP_THREADS, TILE_BYTES, st>>>(
        pl->d_ch_staged + ca, nA, nullptr, tab, (int)ns, stg, lazy, order2, pp);
    else migrate_copy_kernel<true, false><<<(unsigned)nA, CP_THREADS, TILE_BYTES, st>>>(
        pl->d_ch_staged + ca, nA, nullptr, tab, (int)ns, stg, lazy, order2, pp);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
  }
  return ETC_OK;
}

extern "C" etc_status etc_migrate_phase(const etc_plan* pl, const void* const* src_bufs, void* const* dst_bufs,
                                        void* staging, int32_t phases, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl) return ETC_ERR_INVALID_ARG;
  if (pl->lazy && !pl->resolved) {
    // ETC_NO_SYNC plan whose counts are still on the device: grids from the host-side bounds (staged + local chunks
    // together never exceed bound_chunks), the kernels read the real counts and idle CTAs leave at once
    const bool direct = (pl->flags & ETC_ALL_DIRECT) != 0;
    if (!direct && !staging) return ETC_ERR_INVALID_ARG;
    if (direct) phases &= ~ETC_PHASE_UNPACK;
    if (phases == 0) return ETC_OK;
    const long long nb = pl->bound_chunks;
    if (phases == ETC_PHASE_UNPACK)
      return launch_migrate(pl, src_bufs, dst_bufs, staging, phases, (cudaStream_t)stream, pl->d_ptrs, -1, 0, nb, 0, 0, 0, 0,
                            false, 0, pl->d_totals, pl->d_ch1, pl->d_ch2);
    return launch_migrate(pl, src_bufs, dst_bufs, staging, phases, (cudaStream_t)stream, pl->d_ptrs, -1, 0, direct ? 0 : nb, 0,
                          direct ? nb : 0, 0, 0, true, pl->bound_fills, pl->d_totals, pl->d_ch1, pl->d_ch2);
  }
  etc_status rc = ETC_OK;
  const PlanTotals& t = plan_totals(pl, &rc);
  if (rc != ETC_OK) return rc;
  return launch_migrate(pl, src_bufs, dst_bufs, staging, phases, (cudaStream_t)stream, pl->d_ptrs, -1, 0,
                        t.n_chunks_staged, 0, t.n_chunks_local, 0, t.staging_bytes, true, t.n_fills, nullptr,
                        pl->d_ch1, pl->d_ch2);
}

extern "C" etc_status etc_migrate(const etc_plan* pl, const void* const* src_bufs, void* const* dst_bufs, void* staging,
                                  void* stream) {
  return etc_migrate_phase(pl, src_bufs, dst_bufs, staging, ETC_PHASE_ALL, stream);
}

// (f2) one round of state chunking: see rounds.cu
extern "C" etc_status etc_migrate_round(const etc_plan* pl, int32_t round, const void* const* src_bufs,
                                        void* const* dst_bufs, void* staging, int32_t phases, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || round < 0 || (size_t)round >= pl->rounds.size()) return ETC_ERR_INVALID_ARG;
  const RoundRec& r = pl->rounds[round];
  const size_t n_ptrs = ((size_t)(pl->n_old + pl->n_new) * ETC_NUM_KINDS * sizeof(void*) + 255) / 256 * 256 / sizeof(void*);
  return launch_migrate(pl, src_bufs, dst_bufs, staging, phases, (cudaStream_t)stream,
                        pl->d_round_ptrs + n_ptrs * (size_t)round, r.kind, r.ca, r.cb - r.ca, r.la, r.lb - r.la,
                        r.stg_base, r.stg_span, r.sub == 0, plan_totals(pl).n_fills, nullptr,
                        pl->d_rch1 ? pl->d_rch1 + r.ca + r.la : nullptr, pl->d_rch2 ? pl->d_rch2 + r.ca : nullptr);
}
