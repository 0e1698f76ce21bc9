// primitive.cu — the paper's migration primitive as ONE call (PAPER.md:24 "a collective communication primitive"; :86-88
// "takes the previous parallel configuration, the current one and the model state, returns the migrated state"):
// (a1) both layout descriptors, (a2) cost matrix, (a3) sketch, (a4) plan, (a5, a6) pack / unpack / local, submitted
// back to back on the caller's stream with NO host synchronisation anywhere: the layout tables are uploaded behind an
// event, the plan is made with ETC_NO_SYNC (tables sized from host-side bounds, counts stay on the device, the copy
// launches use bound-sized grids whose idle CTAs leave at once).  For a small state the whole reconfiguration then costs
// its kernels plus their launch overheads (the metadata steps are "almost negligible").
#include <future>
#include "etc_internal.h"
#include "plan_types.h"

using namespace etc;

extern "C" etc_status etc_migrate_state(const etc_model_desc* model, const etc_parallel_cfg* old_cfg,
                                        const etc_parallel_cfg* new_cfg, const void* const* src_bufs,
                                        void* const* dst_bufs, void* staging, int64_t staging_bytes,
                                        const uint8_t* d_avail, int32_t flags, etc_plan** plan_out, void* stream) {
  clear_error_detail();
  if (!model || !old_cfg || !new_cfg || !src_bufs || !dst_bufs || staging_bytes < 0) return ETC_ERR_INVALID_ARG;
  if (flags & (ETC_KIND_MAJOR | ETC_NO_SYNC)) return ETC_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  etc_layout *lo = nullptr, *ln = nullptr;
  etc_plan* pl = nullptr;
  char* tmp = nullptr;
  etc_status rc = validate_config(model, old_cfg);      // bad arguments and bad configurations fail before any CUDA call
  if (rc == ETC_OK) rc = validate_config(model, new_cfg);
  if (rc != ETC_OK) return rc;
  // (a1) the two descriptors are independent host-side builds: side by side on two host threads when they are big
  // enough to pay for starting a thread (measured: ~60 us; x64's 2 x 0.4 ms and c4's 2 x 0.12 ms gain, c2's 2 x 51 us
  // would lose, so those are built in turn)
  const long long work = ((long long)old_cfg->tp * old_cfg->pp * old_cfg->dp + (long long)new_cfg->tp * new_cfg->pp * new_cfg->dp) *
                         model->n_layers;
  if (work >= 1024) {
    std::future<etc_status> f_old = std::async(std::launch::async, [&]() { return etc_layout_create(model, old_cfg, &lo); });
    const etc_status rc_new = etc_layout_create(model, new_cfg, &ln);
    rc = f_old.get();
    if (rc == ETC_OK) rc = rc_new;
  } else {
    rc = etc_layout_create(model, old_cfg, &lo);
    if (rc == ETC_OK) rc = etc_layout_create(model, new_cfg, &ln);
  }
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); if (lo) etc_layout_destroy(lo); if (ln) etc_layout_destroy(ln); return ETC_ERR_CUDA; }
  auto done = [&](etc_status r) {
    if (tmp) cudaFreeAsync(tmp, st);
    if (r != ETC_OK && pl) { etc_plan_destroy(pl); pl = nullptr; }
    if (lo) etc_layout_destroy(lo);          // stream-ordered: after every kernel already enqueued that reads the tables
    if (ln) etc_layout_destroy(ln);
    if (r == ETC_OK) { if (plan_out) *plan_out = pl; else etc_plan_destroy(pl); }
    return r;
  };
  if (rc != ETC_OK) return done(rc);
  const int n_old = etc_layout_num_devices(lo), n_new = etc_layout_num_devices(ln), P = n_old > n_new ? n_old : n_new;
  // scratch: overlap [n_new][P] | need [n_new] | hold [P] | local bytes [1] | device map [n_new]
  const size_t o_need = sizeof(int64_t) * (size_t)n_new * P, o_hold = o_need + sizeof(int64_t) * (size_t)n_new,
               o_local = o_hold + sizeof(int64_t) * (size_t)P, o_map = o_local + sizeof(int64_t),
               bytes = o_map + sizeof(int32_t) * (size_t)n_new;
  cudaError_t e = cudaMallocAsync(&tmp, bytes, st);
  if (e != cudaSuccess) { set_error_detail("etc_migrate_state scratch", e); return done(ETC_ERR_CUDA); }
  int64_t* d_ov = reinterpret_cast<int64_t*>(tmp);
  int32_t* d_map = reinterpret_cast<int32_t*>(tmp + o_map);
  rc = etc_cost_matrix(lo, ln, d_ov, reinterpret_cast<int64_t*>(tmp + o_need), reinterpret_cast<int64_t*>(tmp + o_hold), st);   // (a2)
  if (rc == ETC_OK) rc = etc_sketch(d_ov, n_new, P, d_avail, ETC_SKETCH_AUTO, d_map, reinterpret_cast<int64_t*>(tmp + o_local), st);   // (a3)
  if (rc == ETC_OK) rc = etc_plan_create(lo, ln, d_map, flags | ETC_NO_SYNC, &pl, st);              // (a4)
  if (rc != ETC_OK) return done(rc);
  if (!(flags & ETC_ALL_DIRECT)) {
    const int64_t need = (pl->lazy && !pl->resolved) ? pl->bound_staging : plan_totals(pl).staging_bytes;
    if (staging_bytes < need || (need > 0 && !staging)) return done(ETC_ERR_WORKSPACE);
  }
  rc = etc_migrate(pl, src_bufs, dst_bufs, staging, st);                                            // (a5), (a6)
  return done(rc);
}
