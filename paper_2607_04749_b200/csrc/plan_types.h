// plan_types.h — plan-side tables shared by plan.cu (which writes them) and migrate.cu (which reads them).
#pragma once
#include <atomic>
#include <vector>
#include "etc_internal.h"

namespace etc {

struct BlockCount { int64_t slices, chunks, padded, bytes; };   // per (unit, sub-block of pieces); unit = (source device, new rank)
struct UnitBase { int64_t slice0, chunk0, stg0; };
struct PlanTotals {
  int64_t n_slices_staged, n_chunks_staged, staging_bytes, n_slices_local, n_chunks_local;
  int64_t local_bytes, remote_bytes, bad_map;
  int64_t fill_bytes, n_fills;           // zero-filled destination bytes / descriptors (reading A31); added after the scan
  int64_t overflow;                      // ETC_NO_SYNC plans: the tables sized from host-side bounds would not have sufficed
  // kind-major plans: [kind][0] first staged chunk, [1] first staging byte, [2] first local chunk of the kind;
  // entry [ETC_NUM_KINDS] = the totals
  int64_t kind_base[ETC_NUM_KINDS + 1][3];
};

// Shared-memory tile of the copy kernels: one chunk of payload plus slack for the byte-phase re-aligning path, which
// stores row r at r * realign_pitch(row_bytes) + (source address of the row mod 16).
constexpr int TILE_BYTES = ETC_CHUNK_BYTES + 8192;
// tile row pitch of the re-aligning path: the 16-byte slots that can overlap a row of row_bytes at any byte phase
__host__ __device__ __forceinline__ uint32_t realign_pitch(uint32_t row_bytes) { return ((row_bytes + 30u) >> 4) << 4; }
// Rows per chunk of a 2-D slice with rows shorter than ETC_CHUNK_BYTES.  aligned16: every address, pitch and the row
// length are multiples of 16 (the chunk is then staged densely); otherwise the re-aligning path's padded rows must fit.
__host__ __device__ __forceinline__ int rows_per_chunk(int64_t row_bytes, bool aligned16) {
  int rpc = (int)(ETC_CHUNK_BYTES / row_bytes);
  if (!aligned16) {
    const int fit = (int)((TILE_BYTES - 16) / realign_pitch((uint32_t)row_bytes));
    if (fit < rpc) rpc = fit;
  }
  return rpc < 1 ? 1 : rpc;
}

// One copy work item: nrows x row_bytes, at most ETC_CHUNK_BYTES in total (or one row segment of that size).
struct Chunk {
  int64_t src_off, dst_off, stg_off;   // byte offsets inside the source buffer, destination buffer, staging buffer
  int32_t src_stride, dst_stride;      // row pitch in bytes (staging pitch = row_bytes)
  int32_t row_bytes, nrows;
  uint16_t src_buf, dst_buf;           // pointer-table indices: device*4 + kind
  int16_t vec;                         // widest power-of-two access (<= 16 B) every address of the chunk is aligned to
  int16_t pad;                         // 0 in the plan's lists; CHUNK_STAGED marks staged chunks in the ordered launch-1 list
};
constexpr int16_t CHUNK_STAGED = 1;
static_assert(sizeof(Chunk) == 48, "Chunk layout");

// One round of state chunking: a contiguous range of staged chunks whose staging footprint fits the
// caller's bound, plus a share of the same kind's local chunks.
struct RoundRec {
  int64_t ca, cb;                      // staged chunk range [ca,cb)
  int64_t la, lb;                      // local chunk range [la,lb)
  int64_t stg_base, stg_span;          // the round uses staging bytes [stg_base, stg_base + stg_span) of the full layout
  int64_t staged_bytes, local_bytes;   // payload
  int32_t kind, sub, n_sub, pad;
};

}  // namespace etc

struct etc_plan;
namespace etc {
// Call before enqueueing anything that reads the plan's tables on `st`: a stream other than the one the plan was created
// on is made to wait for the plan's last table-writing kernel, and `st` is noted as a reader (frees are ordered after it).
cudaError_t plan_use(const etc_plan* pl, cudaStream_t st);
// The plan's totals on the host.  For an ETC_NO_SYNC plan the first call waits for the plan's kernels and reads them
// back; *rc receives ETC_ERR_BAD_MAP / ETC_ERR_UNRECOVERABLE / ETC_ERR_WORKSPACE if the device found the plan unusable.
const PlanTotals& plan_totals(const etc_plan* pl, etc_status* rc = nullptr);
// plan_order.cu: the address-ordered launch lists of a plan (nA staged, nB local chunks; for an ETC_NO_SYNC plan their
// common bound and the device-side totals)
cudaError_t plan_build_order(etc_plan* pl, long long nA, long long nB, cudaStream_t st, const etc::PlanTotals* lazy = nullptr);
cudaError_t plan_build_round_order(etc_plan* pl, cudaStream_t st);     // after etc_plan_set_rounds filled pl->rounds
}

struct etc_plan {
  int32_t n_old = 0, n_new = 0, P = 0, flags = 0;
  cudaStream_t stream_created_on = nullptr;
  cudaEvent_t ready = nullptr;                     // recorded on stream_created_on after the last table-writing kernel
  mutable etc::StreamSet streams;                  // streams the plan's tables were written / read on (frees are ordered after them)
  etc::PlanTotals totals{};                        // valid once `resolved` (always, unless created with ETC_NO_SYNC)
  // ETC_NO_SYNC: tables sized from upper bounds, counts live on the device until someone asks (plan_totals)
  bool lazy = false;
  std::atomic<bool> resolved{true};                // read without resolve_mu by etc_migrate_phase / etc_migrate_state; totals are read under it
  etc_status resolve_status = ETC_OK;
  int64_t bound_slices = 0, bound_chunks = 0, bound_staging = 0, bound_fills = 0, need_bytes = 0;
  std::mutex resolve_mu;
  void* d_ws = nullptr;                            // blob 1: the tables below up to d_ptrs
  void* d_tb = nullptr;                            // blob 2: slices, first-chunk indices, chunks
  int32_t* d_map = nullptr;
  etc::UnitBase* d_bases = nullptr;
  etc::BlockCount* d_blocks = nullptr;
  int64_t* d_traffic = nullptr;
  etc::PlanTotals* d_totals = nullptr;
  etc_slice* d_sl_staged = nullptr; etc_slice* d_sl_local = nullptr;
  etc::Chunk* d_ch_staged = nullptr; etc::Chunk* d_ch_local = nullptr;
  // address-ordered launch lists (plan_order.cu), or null (launch in list order): d_ch1 = every chunk of launch 1 (staged
  // ones flagged CHUNK_STAGED in `pad`, then packed; the others copied old -> new buffer) sorted by source address,
  // d_ch2 = the staged chunks sorted by destination address for launch 2
  etc::Chunk* d_ch1 = nullptr; etc::Chunk* d_ch2 = nullptr;
  void* d_order_ws = nullptr;
  // the same per round (etc_plan_set_rounds): round i walks d_rch1[ca + la, cb + lb) and d_rch2[ca, cb)
  etc::Chunk* d_rch1 = nullptr; etc::Chunk* d_rch2 = nullptr;
  void* d_round_order_ws = nullptr;
  etc_slice* d_fills = nullptr;                    // zero-fill descriptors (in d_ws; totals.n_fills of them), reading A31
  std::vector<int64_t> old_bytes, new_bytes;       // buffer sizes [dev*4+kind], for argument checks in migrate
  void** d_ptrs = nullptr;                         // [n_old*4] source pointers then [n_new*4] destination pointers
  // state chunking (f2): rounds of bounded staging, set by etc_plan_set_rounds
  std::vector<etc::RoundRec> rounds;
  int64_t round_staging_cap = 0;
  void* d_rounds_ws = nullptr;                     // round records + one pointer table per round
  void** d_round_ptrs = nullptr;
  // host_io.cu: de-duplicated source regions per state kind (src_dev = buffer index), built on first use
  mutable std::vector<etc_slice> h_regions[ETC_NUM_KINDS];
  mutable int64_t h_region_bytes[ETC_NUM_KINDS] = {0, 0, 0, 0};
  mutable bool h_regions_ready = false;
};
