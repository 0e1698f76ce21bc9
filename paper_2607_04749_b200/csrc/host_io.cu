// host_io.cu — host-resident old shards: upload exactly the source bytes the plan reads.
//
// The paper moves only the workload that changes process (Send/Recv carry the slices of the migration
// instructions, Refer moves nothing); an old shard that lives in host memory therefore need not cross PCIe whole.  Every
// slice of the plan names a 2-D region of one old shard buffer (rows x row_bytes at pitch src_stride); this call copies
// those regions, and nothing else, from the host copy of the buffer to the same offsets of its device copy, one
// cudaMemcpy2DAsync (or cudaMemcpyAsync) per region.  Measured on the B200 box: 2-D host-to-device copies run at the
// same 55 GB/s as 1-D copies down to 256-byte rows, so a strided (row-parallel) region costs no more than its payload.
// Regions read by several slices (replicated tensors fanned out to several destinations) are uploaded once.
#include <algorithm>
#include <vector>
#include "etc_internal.h"
#include "plan_types.h"

using namespace etc;

namespace {
struct Region { int64_t off, row_bytes; int32_t stride, nrows, buf; };
inline bool region_less(const Region& a, const Region& b) {
  if (a.buf != b.buf) return a.buf < b.buf;
  if (a.off != b.off) return a.off < b.off;
  if (a.row_bytes != b.row_bytes) return a.row_bytes < b.row_bytes;
  if (a.nrows != b.nrows) return a.nrows < b.nrows;
  return a.stride < b.stride;
}
inline bool region_same(const Region& a, const Region& b) {
  return a.buf == b.buf && a.off == b.off && a.row_bytes == b.row_bytes && a.nrows == b.nrows &&
         (a.nrows == 1 || a.stride == b.stride);
}
}  // namespace

// Build (once per plan) the de-duplicated source regions per state kind, sorted by (buffer, offset), with adjacent
// contiguous 1-D regions of one buffer merged.
static etc_status source_regions(const etc_plan* pl) {
  if (pl->h_regions_ready) return ETC_OK;
  const PlanTotals& t = plan_totals(pl);
  std::vector<etc_slice> sl((size_t)(t.n_slices_staged + t.n_slices_local));
  ETC_CUDA_TRY(cudaStreamSynchronize(pl->stream_created_on));
  if (t.n_slices_staged)
    ETC_CUDA_TRY(cudaMemcpy(sl.data(), pl->d_sl_staged, sizeof(etc_slice) * (size_t)t.n_slices_staged, cudaMemcpyDeviceToHost));
  if (t.n_slices_local)
    ETC_CUDA_TRY(cudaMemcpy(sl.data() + t.n_slices_staged, pl->d_sl_local, sizeof(etc_slice) * (size_t)t.n_slices_local,
                            cudaMemcpyDeviceToHost));
  std::vector<Region> all(sl.size());
  for (size_t i = 0; i < sl.size(); ++i)
    all[i] = Region{sl[i].src_off, sl[i].row_bytes, sl[i].src_stride, sl[i].nrows, sl[i].src_dev * ETC_NUM_KINDS + sl[i].kind};
  std::sort(all.begin(), all.end(), region_less);
  for (int k = 0; k < ETC_NUM_KINDS; ++k) { pl->h_regions[k].clear(); pl->h_region_bytes[k] = 0; }
  for (size_t i = 0; i < all.size(); ++i) {
    if (i && region_same(all[i], all[i - 1])) continue;                      // read by several slices: upload once
    const Region& r = all[i];
    std::vector<etc_slice>& out = pl->h_regions[r.buf % ETC_NUM_KINDS];
    if (!out.empty()) {                                                      // merge contiguous 1-D neighbours
      etc_slice& p = out.back();
      if (r.nrows == 1 && p.nrows == 1 && p.src_dev == r.buf && p.src_off + p.row_bytes == r.off) { p.row_bytes += r.row_bytes; continue; }
    }
    etc_slice e{};
    e.src_off = r.off; e.row_bytes = r.row_bytes; e.src_stride = r.stride; e.nrows = r.nrows; e.src_dev = r.buf;   // src_dev = buffer index here
    out.push_back(e);
  }
  for (int k = 0; k < ETC_NUM_KINDS; ++k)
    for (const etc_slice& e : pl->h_regions[k]) pl->h_region_bytes[k] += (int64_t)e.nrows * e.row_bytes;
  pl->h_regions_ready = true;
  return ETC_OK;
}

extern "C" etc_status etc_upload_sources(const etc_plan* pl, const void* const* h_src_bufs, void* const* d_src_bufs,
                                         int32_t only_kind, int64_t* bytes_out, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !h_src_bufs || !d_src_bufs || only_kind < -1 || only_kind >= ETC_NUM_KINDS) return ETC_ERR_INVALID_ARG;
  etc_status rc = source_regions(pl);
  if (rc != ETC_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  for (int k = 0; k < ETC_NUM_KINDS; ++k) {                   // every buffer a region names must exist on both sides
    if (only_kind >= 0 && k != only_kind) continue;
    for (const etc_slice& e : pl->h_regions[k])
      if (!h_src_bufs[e.src_dev] || !d_src_bufs[e.src_dev]) return ETC_ERR_INVALID_ARG;
  }
  int64_t total = 0;
  for (int k = 0; k < ETC_NUM_KINDS; ++k) {
    if (only_kind >= 0 && k != only_kind) continue;
    for (const etc_slice& e : pl->h_regions[k]) {
      const char* h = static_cast<const char*>(h_src_bufs[e.src_dev]);
      char* d = static_cast<char*>(d_src_bufs[e.src_dev]);
      if (e.nrows == 1) ETC_CUDA_TRY(cudaMemcpyAsync(d + e.src_off, h + e.src_off, (size_t)e.row_bytes, cudaMemcpyHostToDevice, st));
      else ETC_CUDA_TRY(cudaMemcpy2DAsync(d + e.src_off, (size_t)e.src_stride, h + e.src_off, (size_t)e.src_stride,
                                          (size_t)e.row_bytes, (size_t)e.nrows, cudaMemcpyHostToDevice, st));
    }
    total += pl->h_region_bytes[k];
  }
  if (bytes_out) *bytes_out = total;
  return ETC_OK;
}
