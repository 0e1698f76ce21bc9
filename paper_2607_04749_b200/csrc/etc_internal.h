// etc_internal.h — structures shared by the host layout builder and the CUDA kernels of libetc.so.
// Nothing here is shared with oracle/ (the CPU oracle is written separately from the paper).
#pragma once
#include <cstdint>
#include <mutex>
#include <vector>
#include <cuda_runtime.h>
#include "../../include/etc.h"

namespace etc {

// Split type of a logical tensor (PAPER.md:199 replaced by an explicit type, reading A8).
enum Split : int32_t { REPL = 0, COL = 1, ROW = 2, COL2 = 3, QKV = 4 };

// Piece flags
enum : uint16_t {
  PF_POST_COPY = 1,   // tied word_embeddings replica held by the last PP stage (reading A11)
  PF_SOLE_INST = 2,   // the tensor is held by exactly one PP stage in this layout
  PF_DP_SHARDED = 8,  // kind is sharded over DP (distributed optimizer, reading A14)
};

// One index rectangle [r0,r0+nr) x [c0,c0+nc) of a logical tensor held in the buffer of (dev, kind).
// Local (shard) coordinates: element (r0,c0) is element (lrow0, lcol0) of the TP shard, whose row length is W.
// [f0,f1) is the flat range of the SHARD (shard-relative, in elements) that this buffer holds; all pieces of one
// (dev, group) carry the same [f0,f1).
struct Piece {
  int32_t dev;        // logical device / rank in this layout
  int32_t grp;        // kind * n_tensors + logical tensor id
  int32_t r0, nr, c0, nc;
  int32_t lrow0, lcol0;
  int32_t W;          // row pitch in elements inside the buffer
  int16_t s, r, d;    // PP stage, TP rank, DP rank of dev
  uint16_t flags;
  int16_t rep, rbase; // the TP ranks [rbase, rbase + rep) of stage s hold these elements: rep = 1 TP-sharded, rep = tp
                      // replicated tensor, rep = tp / n_kv K or V head under KV-head replication (reading A30)
  int64_t boff;       // byte offset of element (r0,c0) inside the buffer of (dev, kind)
  int64_t f0, f1;
};
static_assert(sizeof(Piece) == 72, "Piece layout");

struct DeviceTables {            // device memory
  const Piece* pieces;           // sorted by (dev, grp, local order)
  const int32_t* dev_start;      // [n_dev + 1]
  const int32_t* first;          // [n_dev][n_grp]: index of the first piece of (dev, grp) or -1
  const uint32_t* ltmask;        // [n_dev][mask_words]: bit t set if dev holds any piece of logical tensor t
  const int32_t* kind_start;     // [n_dev][ETC_NUM_KINDS + 1]: piece range of each state kind on dev (pieces are kind-major)
  int32_t n_dev, n_grp, n_tensors, mask_words;
  int32_t n_pieces;
  int32_t tp, pp, dp;
  int32_t elem_bytes[ETC_NUM_KINDS];
};

// The streams on which kernels reading an object's device tables have been enqueued.  The tables are released with a
// stream-ordered free; join() returns the most recently used stream after making it wait (by event) for everything
// enqueued so far on every other noted stream, so the free is ordered after all readers.  A NULL cudaStream_t is the
// legacy default stream and is a stream like any other here (it must not be mistaken for "never used").
struct StreamSet {
  std::vector<cudaStream_t> used;
  std::mutex mu;                   // note() is called through const handles from any host thread
  void note(cudaStream_t st) {
    std::lock_guard<std::mutex> lock(mu);
    for (size_t i = 0; i < used.size(); ++i)
      if (used[i] == st) { used.erase(used.begin() + (long)i); break; }
    used.push_back(st);
  }
  cudaStream_t join(cudaStream_t fallback) {
    std::lock_guard<std::mutex> lock(mu);
    if (used.empty()) return fallback;
    cudaStream_t last = used.back();
    for (size_t i = 0; i + 1 < used.size(); ++i) {
      cudaEvent_t e;
      if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { (void)cudaGetLastError(); continue; }
      if (cudaEventRecord(e, used[i]) == cudaSuccess) cudaStreamWaitEvent(last, e, 0);
      cudaEventDestroy(e);
      (void)cudaGetLastError();
    }
    return last;
  }
};

}  // namespace etc

struct etc_layout {
  etc_model_desc model;
  etc_parallel_cfg cfg;
  etc::DeviceTables t;                    // device pointers + sizes
  int64_t* h_buffer_bytes = nullptr;      // [n_dev][4] host
  int32_t max_dev_pieces = 0;             // largest piece count of one device
  int32_t vocab_rows = 0;                 // rows of the embedding tensors in this layout (padded vocabulary, reading A31)
  int32_t lm_head_id = -1;                // logical tensor id of lm_head (-1: tied); word_embeddings is tensor 0
  int32_t n_emb_pieces = 0;               // pieces of the embedding tensors (upper bound of the zero-fill list)
  std::vector<int32_t> grp_pieces;        // [n_grp] pieces of each (kind, tensor) group over all devices (plan size bounds)
  std::vector<int32_t> stage_first;       // [pp + 1] first layer of each pipeline stage (stage s holds [s], [s+1]) 
  bool aligned16 = true;                  // every piece of a tensor with more than one column has its offset, pitch, column
                                          // range and held flat range at multiples of 16 B: every STRIDED slice (rows that
                                          // do not merge into one run) is then 16-byte aligned and chunked by payload alone
  int64_t total_bytes = 0;                // sum of all buffer sizes
  void* d_blob = nullptr;                 // one allocation holding all device tables
  cudaEvent_t ready = nullptr;            // recorded behind the upload of d_blob (layout_use waits for it)
  mutable etc::StreamSet streams;         // streams that kernels reading the tables were enqueued on
};

// ---- error plumbing
namespace etc {
void set_error_detail(const char* what, cudaError_t e);
void set_error_text(const char* text);                 // a detail that is not a CUDA error (read by etc_last_error_detail)
void clear_error_detail();
void count_launch(int n = 1);
int current_device();
// Makes the library's device (etc_init) current for the lifetime of the guard and restores the caller's device after.
struct DeviceGuard {
  int prev = -1; bool switched = false; cudaError_t err = cudaSuccess;
  DeviceGuard() {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != current_device()) { err = cudaSetDevice(current_device()); switched = err == cudaSuccess; }
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
etc_status validate_config(const etc_model_desc* m, const etc_parallel_cfg* c);   // host-only checks of etc_layout_create
cudaError_t layout_use(const etc_layout* L, cudaStream_t st);   // `st` waits for the tables' upload; noted as a reader
// xfer.cu: metadata transfers as kernels on the caller's stream, so that they never queue behind bulk DMA transfers
cudaError_t write_small(void* d_dst, const void* h_src, size_t bytes, cudaStream_t st);      // host -> device via kernel parameters
cudaError_t copy_by_kernel(void* dst, const void* src, size_t bytes, cudaStream_t st);       // device / pinned host, either way
std::mutex& pinned_scratch_mutex();                   // hold it while the scratch is in use
void* pinned_scratch(size_t bytes);                   // grow-only pinned buffer (nullptr on failure)
}
#define ETC_CUDA_TRY(expr)                                          \
  do {                                                              \
    cudaError_t _e = (expr);                                        \
    if (_e != cudaSuccess) {                                        \
      etc::set_error_detail(#expr, _e);                             \
      return ETC_ERR_CUDA;                                          \
    }                                                               \
  } while (0)
