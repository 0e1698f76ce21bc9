// copy_paths.cuh — device-side copy routines of the pack / unpack / local kernels (migrate.cu): one CTA copies one chunk,
// nrows x row_bytes (<= ETC_CHUNK_BYTES of payload) with independent row pitches on the two sides, through a shared-
// memory tile.  Pure byte movement (PAPER.md:197 pack / unpack, :195 Refer).  Which path a chunk takes:
//
//   16-byte aligned chunks (every address, pitch and the row length a multiple of 16):
//     * rows >= TMA_MIN_ROW, or one contiguous run: TMA bulk copies issued by ONE warp — cp.async.bulk global -> shared
//       per row into a dense tile (one copy if the source side is dense), mbarrier wait, cp.async.bulk shared -> global per
//       row (one copy if the destination side is dense).
//     * shorter rows: the DENSE side still moves as one bulk copy (pack: staging is dense; unpack: staging is dense) and
//       only the STRIDED side is handled per 16-byte vector by all 256 threads: gather with cp.async (LDGSTS, the whole
//       chunk in flight at once), scatter with st.global from the tile.  A strided -> strided chunk (local copy) is
//       gathered with cp.async and scattered from the tile.
//   chunks that are not 16-byte aligned (odd hidden sizes, unaligned distributed-optimizer cuts; alignment 1, 2, 4 or 8):
//     * the byte-phase re-aligning path: every source row is loaded as the 16-byte ALIGNED slots that cover it (cp.async
//       16 B; up to 15 bytes before and after the row are read and dropped — inside the 16-byte granule of the buffer,
//       whose base is 16-byte aligned), row r of the tile starts at the row's phase (address mod 16), and every aligned
//       16-byte slot of the DESTINATION row is assembled from the two aligned 16-byte tile slots that cover it (two
//       LDS.128, word selects, funnel shifts) and written with one 16-byte store; only the ragged ends of a row use
//       narrow stores.
#pragma once
#include <cstdint>
#include "plan_types.h"

namespace etc {

constexpr int CP_THREADS = 256;
constexpr int TMA_MIN_ROW = 1024;                       // below this, per-row bulk copies issued by one warp lose to the
                                                        // 256-thread short-row path (measured: 512-byte rows strided on both
                                                        // sides 5.7 vs 6.5 TB/s; equal from 1 KB rows on)

template <typename V> __device__ __forceinline__ V ld_stream(const V* p) { return __ldcs(p); }
template <typename V> __device__ __forceinline__ void st_stream(V* p, const V& v) { __stcs(p, v); }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- cp.async (LDGSTS)
__device__ __forceinline__ void cp_async16(void* smem, const void* g) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit_wait() {
  asm volatile("cp.async.commit_group;" ::: "memory");
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// ---- TMA bulk copies + mbarrier (sm_100a)
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
__device__ __forceinline__ void bulk_store_drain() {
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");      // the tile must outlive the reads of the bulk stores
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

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
  bulk_store_drain();
}

// ---- short 16-byte aligned rows (row_bytes < TMA_MIN_ROW, nrows > 1): all CP_THREADS threads.
// Vector v of the dense tile = (row v / vpr, 16-byte column v % vpr); multiply-high reciprocal, exact for v < 2^32 / vpr.
struct RowDiv {
  uint32_t vpr, magic;
  __device__ __forceinline__ explicit RowDiv(uint32_t vpr_) : vpr(vpr_), magic((uint32_t)((0x100000000ull + vpr_ - 1) / vpr_)) {}
  __device__ __forceinline__ void split(uint32_t v, uint32_t& row, uint32_t& col) const {
    row = vpr == 1 ? v : __umulhi(v, magic); col = v - row * vpr;
  }
};

__device__ __forceinline__ void short_rows_copy_chunk(char* tile, uint64_t* bar, const char* __restrict__ src,
                                                      char* __restrict__ dst, int nrows, uint32_t row_bytes, uint32_t sp,
                                                      uint32_t dp) {
  const uint32_t total = row_bytes * (uint32_t)nrows, nvec = total >> 4;
  const RowDiv rd(row_bytes >> 4);
  const bool src_dense = sp == row_bytes, dst_dense = dp == row_bytes;
  const uint32_t tid = threadIdx.x;
  // ---- in: global -> dense tile
  if (src_dense) {                                     // one bulk copy (unpack: the staging side)
    if (tid == 0) { mbar_init(bar, 1); mbar_expect_tx(bar, total); bulk_g2s(tile, src, total, bar); }
    __syncthreads();                                   // the barrier is initialised before anyone polls it
    mbar_wait(bar, 0);
  } else {                                             // gather: every 16-byte vector of the chunk in flight at once
    for (uint32_t v = tid; v < nvec; v += CP_THREADS) {
      uint32_t row, col; rd.split(v, row, col);
      cp_async16(tile + ((size_t)v << 4), src + (size_t)row * sp + ((size_t)col << 4));
    }
    cp_async_commit_wait();
  }
  // ---- out: dense tile -> global
  if (dst_dense) {                                     // one bulk copy (pack: the staging side)
    fence_proxy_async();                               // this thread's tile writes become visible to the async proxy
    __syncthreads();
    if (tid == 0) { bulk_s2g(dst, tile, total); bulk_store_drain(); }
  } else {                                             // scatter; a thread re-reads exactly the vectors it loaded itself
    for (uint32_t v = tid; v < nvec; v += CP_THREADS) {
      uint32_t row, col; rd.split(v, row, col);
      st_stream(reinterpret_cast<uint4*>(dst + (size_t)row * dp) + col, *reinterpret_cast<const uint4*>(tile + ((size_t)v << 4)));
    }
  }
}

// ---- byte-phase re-aligning path: chunks whose addresses are only 1-, 2-, 4- or 8-byte aligned.  `vec` = that alignment
// (every address of the chunk and the row length are multiples of it).  Needs nrows * realign_pitch(row_bytes) <=
// TILE_BYTES - 16, which the plan guarantees by cutting such slices into chunks of fewer rows (rows_per_chunk).
__device__ __forceinline__ void realign_copy_chunk(char* tile, const char* __restrict__ src, char* __restrict__ dst, int nrows,
                                                   uint32_t row_bytes, uint32_t sp, uint32_t dp, int vec) {
  const uint32_t RP = realign_pitch(row_bytes), S = RP >> 4;
  const uint32_t slots = S * (uint32_t)nrows;
  const RowDiv rd(S);
  const uintptr_t s0 = reinterpret_cast<uintptr_t>(src), d0 = reinterpret_cast<uintptr_t>(dst);
  // ---- in: the aligned 16-byte slots covering each source row
  for (uint32_t j = threadIdx.x; j < slots; j += CP_THREADS) {
    uint32_t row, k; rd.split(j, row, k);
    const uintptr_t sa = s0 + (uintptr_t)row * sp;
    const uint32_t sphase = (uint32_t)(sa & 15);
    if ((k << 4) >= sphase + row_bytes) continue;       // slot lies behind the row
    cp_async16(tile + (size_t)row * RP + (k << 4), reinterpret_cast<const char*>(sa - sphase) + (k << 4));
  }
  cp_async_commit_wait();
  __syncthreads();
  // ---- out: the aligned 16-byte slots of each destination row, assembled from the tile at the source's phase
  for (uint32_t j = threadIdx.x; j < slots; j += CP_THREADS) {
    uint32_t row, k; rd.split(j, row, k);
    const uint32_t sphase = (uint32_t)((s0 + (uintptr_t)row * sp) & 15);
    const uintptr_t da = d0 + (uintptr_t)row * dp;
    const uint32_t dphase = (uint32_t)(da & 15);
    const int32_t lo = max((int32_t)(k << 4) - (int32_t)dphase, 0);                       // row bytes [lo, hi) of this slot
    const int32_t hi = min((int32_t)(k << 4) - (int32_t)dphase + 16, (int32_t)row_bytes);
    if (hi <= lo) continue;
    const uint32_t toff = row * RP + sphase + (uint32_t)lo;     // tile offset of the first byte this slot needs
    const char* t = tile + toff;
    char* d = reinterpret_cast<char*>(da) + lo;
    if (hi - lo == 16) {
      // the 16 bytes [t, t+16) out of the two ALIGNED 16-byte tile slots that cover them: two conflict-free LDS.128
      // (five LDS.32 at a 16-byte lane stride would be 4-way bank conflicts each), then words W[wi .. wi+4], wi = o / 4,
      // picked by two rounds of selects (no divergence) and funnel-shifted by the byte remainder
      const uint4* a = reinterpret_cast<const uint4*>(tile + (toff & ~15u));
      const uint4 q0 = a[0];
      const uint32_t o = toff & 15u;
      uint4 q = q0;
      if (o != 0) {
        const uint4 q1 = a[1];
        const uint32_t sh = (o & 3u) << 3;
        const bool b1 = (o & 8u) != 0, b0 = (o & 4u) != 0;
        const uint32_t v0 = b1 ? q0.z : q0.x, v1 = b1 ? q0.w : q0.y, v2 = b1 ? q1.x : q0.z, v3 = b1 ? q1.y : q0.w,
                       v4 = b1 ? q1.z : q1.x, v5 = b1 ? q1.w : q1.y;
        const uint32_t u0 = b0 ? v1 : v0, u1 = b0 ? v2 : v1, u2 = b0 ? v3 : v2, u3 = b0 ? v4 : v3, u4 = b0 ? v5 : v4;
        q.x = __funnelshift_r(u0, u1, sh); q.y = __funnelshift_r(u1, u2, sh);
        q.z = __funnelshift_r(u2, u3, sh); q.w = __funnelshift_r(u3, u4, sh);
      }
      st_stream(reinterpret_cast<uint4*>(d), q);
    } else {                                            // ragged end of the row: the chunk's own alignment
      const int32_t n = hi - lo;
      if (vec >= 8) for (int32_t x = 0; x < n; x += 8) st_stream(reinterpret_cast<uint2*>(d + x), *reinterpret_cast<const uint2*>(t + x));
      else if (vec == 4) for (int32_t x = 0; x < n; x += 4) st_stream(reinterpret_cast<uint32_t*>(d + x), *reinterpret_cast<const uint32_t*>(t + x));
      else if (vec == 2) for (int32_t x = 0; x < n; x += 2) st_stream(reinterpret_cast<uint16_t*>(d + x), *reinterpret_cast<const uint16_t*>(t + x));
      else for (int32_t x = 0; x < n; ++x) d[x] = t[x];
    }
  }
}

// One chunk through the path its shape and alignment select.  All threads of the CTA call this.
template <int MIN_ROW = TMA_MIN_ROW>
__device__ __forceinline__ void copy_one_chunk(char* tile, uint64_t* bar, const char* src, char* dst, int nrows,
                                               uint32_t row_bytes, uint32_t sp, uint32_t dp, int vec) {
  if (vec == 16) {
    if (nrows == 1 || row_bytes >= (uint32_t)MIN_ROW) {
      if (threadIdx.x < 32) tma_copy_chunk(tile, bar, src, dst, nrows, row_bytes, sp, dp);
    } else {
      short_rows_copy_chunk(tile, bar, src, dst, nrows, row_bytes, sp, dp);
    }
    return;
  }
  realign_copy_chunk(tile, src, dst, nrows, row_bytes, sp, dp, vec);
}

}  // namespace etc
