// migrate.cu — (a5) pack, (a6) unpack + local: the HBM-bound hot loop ("The states can be packed to the
// instructions when Send and then unpacked to update the corresponding state after migration"; :195 Refer).
//
// Pure byte movement: a batched gather/scatter over the plan's chunk list.  One CTA copies one chunk (<= 64 KB):
// nrows x row_bytes with independent row pitches on the two sides.
//   * 16-byte aligned chunks with rows >= 512 B (or one contiguous run) go through shared memory with TMA bulk copies:
//     one warp issues cp.async.bulk global -> shared for every row (one mbarrier collects the bytes), then
//     cp.async.bulk shared -> global for every row.  A row-parallel (strided) slice is thus gathered into a dense
//     64 KB tile and written back out with the other side's pitch; three CTAs per SM keep ~192 KB in flight per SM.
//     Measured 6.8-6.9 TB/s against 6.5-6.7 TB/s for the vector path on the same chunk lists.
//   * chunks that are only 4- or 8-byte aligned are staged through the same tile with cp.async (LDGSTS), all loads of
//     the chunk in flight at once; rows >= 256 B are re-aligned on the way (16-byte loads into a tile row that starts at
//     the source's phase modulo 16, 16-byte stores assembled from narrow shared-memory reads): 6.5 TB/s on a layout
//     with half its bytes misaligned, against 5.4 TB/s with register staging.
//   * everything else (16-byte aligned rows < 512 B, or 1- / 2-byte alignment) takes the vector path: the widest
//     aligned access, streaming loads/stores, four independent vectors in flight per thread.
// Two launches per migration:
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

// ---- cp.async staged path for chunks that are only 4- or 8-byte aligned (odd hidden sizes, unaligned distributed-
// optimizer cuts).  With register staging a thread keeps 4 narrow loads in flight and the CTA a few KB; here every
// thread issues ALL its loads of the chunk as cp.async (LDGSTS) into the 64 KB tile, so the whole chunk is in flight,
// as on the TMA path, and writes its own elements out again after its wait_group (no block barrier: a thread reads
// back only what it loaded).  ncu on a layout with 52 % of the bytes misaligned: register path 27 % warps active,
// stalled on long_scoreboard, 4.5 TB/s on the misaligned share.
template <int VB> __device__ __forceinline__ void cp_async(void* smem, const void* g) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(g), "n"(VB) : "memory");
}
template <typename V>
__device__ __forceinline__ void staged_copy_chunk(char* __restrict__ tile, const char* __restrict__ src, char* __restrict__ dst,
                                                  int nrows, uint32_t row_bytes, uint32_t src_pitch, uint32_t dst_pitch) {
  constexpr uint32_t VB = (uint32_t)sizeof(V);
  const uint32_t vpr = row_bytes / VB, total = vpr * (uint32_t)nrows;
  const uint32_t magic = (uint32_t)((0x100000000ull + vpr - 1) / vpr);
  for (uint32_t i = threadIdx.x; i < total; i += CP_THREADS) {
    const uint32_t row = (nrows == 1) ? 0 : (vpr == 1 ? i : __umulhi(i, magic)), col = i - row * vpr;
    cp_async<(int)VB>(tile + (size_t)i * VB, src + (size_t)row * src_pitch + (size_t)col * VB);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  for (uint32_t i = threadIdx.x; i < total; i += CP_THREADS) {
    const uint32_t row = (nrows == 1) ? 0 : (vpr == 1 ? i : __umulhi(i, magic)), col = i - row * vpr;
    st_stream(reinterpret_cast<V*>(dst + (size_t)row * dst_pitch + (size_t)col * VB), *reinterpret_cast<const V*>(tile + (size_t)i * VB));
  }
}

// Re-aligning variant for rows >= 256 B: 16-byte loads AND 16-byte stores although source and destination disagree
// modulo 16.  Row r of the tile starts at r*RP + (address of its SOURCE row mod 16), so every 16-byte slot of the tile
// that lies wholly inside the row is one 16-byte cp.async from an aligned source address; on the way out every
// 16-byte slot of the DESTINATION row is assembled from 16/sizeof(V) narrow shared-memory reads (the tile is V-aligned
// there, not 16-byte aligned) and written with one 16-byte store.  Only the ragged ends of a row use the narrow width.
// The per-row slack (<= 32 B) fits the tile's 8 KB margin because such a chunk has at most 256 rows.
constexpr int TILE_BYTES = ETC_CHUNK_BYTES + 8192;
constexpr uint32_t REALIGN_MIN_ROW = 256;
template <typename V>
__device__ __forceinline__ void staged_copy_realign(char* __restrict__ tile, const char* __restrict__ src, char* __restrict__ dst,
                                                    int nrows, uint32_t row_bytes, uint32_t src_pitch, uint32_t dst_pitch) {
  constexpr uint32_t VB = (uint32_t)sizeof(V);
  const uint32_t RP = (row_bytes + 31u) & ~15u;                 // >= row_bytes + 16
  const uint32_t S = RP / 16u, slots = S * (uint32_t)nrows;
  const uint32_t magic_s = (uint32_t)((0x100000000ull + S - 1) / S);
  const uint32_t sphase0 = (uint32_t)(reinterpret_cast<uintptr_t>(src) & 15), dphase0 = (uint32_t)(reinterpret_cast<uintptr_t>(dst) & 15);
  for (uint32_t j = threadIdx.x; j < slots; j += CP_THREADS) {
    const uint32_t row = nrows == 1 ? 0 : __umulhi(j, magic_s), k = j - row * S;
    const uint32_t sphase = (sphase0 + row * src_pitch) & 15u;
    const uint32_t lo = max(16u * k, sphase), hi = min(16u * k + 16u, sphase + row_bytes);
    if (hi <= lo) continue;
    const char* g = src + (size_t)row * src_pitch + (lo - sphase);
    char* t = tile + (size_t)row * RP + lo;
    if (hi - lo == 16u) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(t)), "l"(g) : "memory");
    else for (uint32_t x = 0; x < hi - lo; x += VB) cp_async<(int)VB>(t + x, g + x);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  for (uint32_t j = threadIdx.x; j < slots; j += CP_THREADS) {
    const uint32_t row = nrows == 1 ? 0 : __umulhi(j, magic_s), k = j - row * S;
    const uint32_t sphase = (sphase0 + row * src_pitch) & 15u, dphase = (dphase0 + row * dst_pitch) & 15u;
    const uint32_t lo = max(16u * k, dphase), hi = min(16u * k + 16u, dphase + row_bytes);
    if (hi <= lo) continue;
    const uint32_t x0 = lo - dphase;                             // offset inside the row
    char* d = dst + (size_t)row * dst_pitch + x0;
    const char* t = tile + (size_t)row * RP + sphase + x0;       // V-aligned
    if (hi - lo == 16u) {
      union { uint4 q; V v[16 / VB]; } u;
#pragma unroll
      for (uint32_t i = 0; i < 16 / VB; ++i) u.v[i] = reinterpret_cast<const V*>(t)[i];
      st_stream(reinterpret_cast<uint4*>(d), u.q);
    } else {
      for (uint32_t x = 0; x < hi - lo; x += VB) st_stream(reinterpret_cast<V*>(d + x), *reinterpret_cast<const V*>(t + x));
    }
  }
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

// ---- TMA bulk path (sm_100a): cp.async.bulk + mbarrier, issued by one warp
constexpr int TMA_MIN_ROW = 512;          // below this the per-row issue cost outweighs the gain (measured: 256 B rows lose)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "ETC_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra ETC_DONE;\n"
      "bra ETC_WAIT;\n"
      "ETC_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem, const void* g, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem)),
               "l"(g), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* g, const void* smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(g), "r"(smem_u32(smem)), "r"(bytes) : "memory");
}

// One warp: gather nrows x row_bytes (<= ETC_CHUNK_BYTES, everything a multiple of 16 bytes) into the dense tile, then
// scatter it.  A side whose pitch equals row_bytes is one bulk copy; otherwise the lanes issue one bulk copy per row.
__device__ __forceinline__ void tma_copy_chunk(char* tile, uint64_t* bar, const char* __restrict__ src, char* __restrict__ dst,
                                               int nrows, uint32_t row_bytes, uint32_t sp, uint32_t dp) {
  const int lane = threadIdx.x;
  const uint32_t total = row_bytes * (uint32_t)nrows;
  if (lane == 0) { mbar_init(bar, 1); mbar_expect_tx(bar, total); }
  __syncwarp();
  if (nrows == 1 || sp == row_bytes) { if (lane == 0) bulk_g2s(tile, src, total, bar); }
  else for (int r = lane; r < nrows; r += 32) bulk_g2s(tile + (size_t)r * row_bytes, src + (size_t)r * sp, row_bytes, bar);
  mbar_wait(bar, 0);
  if (nrows == 1 || dp == row_bytes) { if (lane == 0) bulk_s2g(dst, tile, total); }
  else for (int r = lane; r < nrows; r += 32) bulk_s2g(dst + (size_t)r * dp, tile + (size_t)r * row_bytes, row_bytes);
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");      // the tile must outlive the reads of the bulk stores
}

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
template <bool UNPACK, bool PARAM_PTRS>
__global__ void __launch_bounds__(CP_THREADS)
migrate_copy_kernel(const Chunk* __restrict__ chA, long long nA, const Chunk* __restrict__ chB,
                    const void* const* __restrict__ tab, int ns, char* __restrict__ staging,
                    const __grid_constant__ PtrParams pp) {
  extern __shared__ __align__(128) char tile[];                 // TILE_BYTES: TMA path and cp.async staged paths
  __shared__ uint64_t bar;
  const long long b = blockIdx.x;
  const bool staged = b < nA;
  const Chunk c = staged ? chA[b] : chB[b - nA];
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
  if (c.vec == 16 && (c.nrows == 1 || c.row_bytes >= TMA_MIN_ROW)) {
    if (threadIdx.x < 32) tma_copy_chunk(tile, &bar, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp);
    return;
  }
  if (c.vec == 8 || c.vec == 4) {
    const bool wide = (uint32_t)c.row_bytes >= REALIGN_MIN_ROW;
    if (c.vec == 8) { if (wide) staged_copy_realign<uint2>(tile, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp);
                      else staged_copy_chunk<uint2>(tile, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp); }
    else { if (wide) staged_copy_realign<unsigned int>(tile, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp);
           else staged_copy_chunk<unsigned int>(tile, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp); }
    return;
  }
  copy_dispatch(c.vec, src, dst, c.nrows, (uint32_t)c.row_bytes, sp, dp);
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
                    const __grid_constant__ PtrParams pp) {
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
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
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
                                 long long la, long long nB, int64_t stg_base, int64_t stg_need, bool with_fills) {
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
        pl->d_ch_staged + ca, nA, pl->d_ch_local + la, tab, (int)ns, stg, pp);
    else migrate_copy_kernel<false, false><<<(unsigned)(nA + nB), CP_THREADS, TILE_BYTES, st>>>(
        pl->d_ch_staged + ca, nA, pl->d_ch_local + la, tab, (int)ns, stg, pp);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
  }
  if ((phases & ETC_PHASE_PACK) && with_fills && pl->totals.n_fills > 0) {      // reading A31: bytes with no source
    const dim3 grid((unsigned)pl->totals.n_fills, FILL_SPLIT);
    if (in_params) migrate_fill_kernel<true><<<grid, CP_THREADS, 0, st>>>(pl->d_fills, tab, (int)ns, only_kind, pp);
    else migrate_fill_kernel<false><<<grid, CP_THREADS, 0, st>>>(pl->d_fills, tab, (int)ns, only_kind, pp);
    ETC_CUDA_TRY(cudaGetLastError());
    count_launch();
  }
  if ((phases & ETC_PHASE_UNPACK) && nA > 0) {
    if (in_params) migrate_copy_kernel<true, true><<<(unsigned)nA, CP_THREADS, TILE_BYTES, st>>>(
        pl->d_ch_staged + ca, nA, nullptr, tab, (int)ns, stg, pp);
    else migrate_copy_kernel<true, false><<<(unsigned)nA, CP_THREADS, TILE_BYTES, st>>>(
        pl->d_ch_staged + ca, nA, nullptr, tab, (int)ns, stg, pp);
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
                        t.n_chunks_staged, 0, t.n_chunks_local, 0, t.staging_bytes, true);
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
                        r.stg_base, r.stg_span, r.sub == 0);
}
