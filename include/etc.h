/*
 * etc.h — C ABI of libetc.so: the data-parallel hot path of ETC's checkpoint-free model-state migration
 * (arxiv/paper_2607_04749, "ETC"; citations below are PAPER.md line numbers and DESIGN.md readings A1-A31).
 *
 * The paper's primitive takes the previous parallel configuration, the current one and the model state, and
 * returns the migrated state.  Here that is four steps, each a call:
 *
 *   etc_layout_create   (a1)  (model_desc, parallel_cfg) -> index rectangles of every state tensor on every device
 *                             (PAPER.md:106 workload abstraction, :110 "each device can derive its workload following
 *                             these rules", :199 TP slices)
 *   etc_cost_matrix     (a2)  old x new index-range intersection -> overlap / need / hold, the paper's cost matrix is
 *                             c[n][o] = need[n] - overlap[n][o]  (worked example :108)
 *   etc_sketch          (a3)  device-side assignment search -> device_map (Eq. 1-4, Algorithm 1)
 *   etc_plan_create     (a4)  Send/Recv/Refer instruction lists as a slice table, coalesced per (src,dst) pair
 *
 *   etc_migrate      (a5,a6)  pack -> staging -> unpack, plus direct copies of what stays on its device
 *                             ("packed to the instructions when Send and then unpacked")
 *
 * All virtual devices' shard buffers live in ONE GPU's memory; the interconnect hop between pack and unpack is the
 * identity (unpack reads the staging buffer pack wrote).  Every step runs in CUDA kernels for sm_100a; there is no CPU
 * fallback: without a CUDA device every compute entry point returns ETC_ERR_CUDA.
 *
 * Conventions
 *  - Plain C types only.  "device pointer" = CUDA device memory of the current device; "host pointer" = ordinary memory.
 *  - `stream` is a cudaStream_t passed as void* (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream.
 *  - Ownership: the caller owns every data buffer, the staging buffer and the output matrices.  The library owns only
 *    etc_layout / etc_plan objects (and their device-side tables), released by the matching destroy call.
 *  - Errors: a negative etc_status; nothing is written to the outputs on error.  etc_last_error_detail() returns a
 *    static/thread-local string with the CUDA error text after ETC_ERR_CUDA.
 *  - Old logical rank j sits on physical device j; new logical rank n is placed on physical device
 *    device_map[n]; P = max(n_old, n_new) physical devices exist.
 *  - Device id = r + tp*(d + dp*s) for TP rank r, DP rank d, PP stage s (reading A9).
 */
#ifndef ETC_H_
#define ETC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef int32_t etc_status;
enum {
  ETC_OK = 0,
  ETC_ERR_INVALID_ARG = -1,  /* null pointer, non-positive size, unknown enum, misaligned buffer */
  ETC_ERR_INDIVISIBLE = -2,  /* n_layers % pp, n_kv_heads % tp (tp <= n_kv_heads), ffn_hidden % tp or vocab % tp != 0
                                 */
  ETC_ERR_MISMATCH = -3,     /* old and new layouts describe different models / kinds */
  ETC_ERR_BAD_MAP = -4,      /* device_map not injective or out of [0,P) */
  ETC_ERR_WORKSPACE = -5,    /* problem larger than the kernel's on-chip workspace (sketch: P > ETC_SKETCH_MAX_P) */
  ETC_ERR_UNSUPPORTED = -6,  /* tp > n_kv_heads where KV-head replication (reading A30) cannot be formed: tp is not a
                                multiple of n_kv_heads, or tp/n_kv_heads does not divide the q heads of a KV group */
  ETC_ERR_CUDA = -7,         /* a CUDA call failed, or no CUDA device */
  ETC_ERR_UNRECOVERABLE = -8 /* some needed bytes have no surviving source (every replica failed, reading A26) */
};

enum { ETC_GPT = 0, ETC_LLAMA = 1 };                 /* etc_model_desc.style */
enum { ETC_BF16 = 2, ETC_FP32 = 4 };                 /* etc_model_desc.param_dtype = element size in bytes */
enum { ETC_QKV_GROUPED = 0, ETC_QKV_BLOCKED = 1 };   /* etc_model_desc.qkv_order */
enum { ETC_K_PARAM = 1, ETC_K_MASTER = 2, ETC_K_ADAM_M = 4, ETC_K_ADAM_V = 8 };   /* kinds bitmask; kind index 0..3 */
#define ETC_NUM_KINDS 4
#define ETC_SKETCH_MAX_P 2048

/* Logical model: the tensors a TP=PP=DP=1 run would hold (table of tensors and split types).
 * ETC_GPT: LayerNorm weight+bias, linear biases, learned position embeddings; ETC_LLAMA: RMSNorm, no bias, SwiGLU. */
typedef struct {
  int32_t style;
  int32_t n_layers, hidden, n_q_heads, n_kv_heads, head_dim, ffn_hidden, vocab, max_pos;
  int32_t tied_embeddings;   /* 1: the output layer shares word_embeddings (replica on the last PP stage if pp > 1) */
  int32_t param_dtype;       /* ETC_BF16 | ETC_FP32: element size of kind PARAM; MASTER / ADAM_M / ADAM_V are fp32 */
  int32_t kinds;             /* bitmask of state kinds present */
  int32_t qkv_order;         /* logical row order of the fused QKV weight / bias (f3, readings A10, A29):
                                ETC_QKV_GROUPED: per KV group its q heads, then K, then V (Megatron's fused layout);
                                ETC_QKV_BLOCKED: [Q; K; V], all q heads, then all k heads, then all v heads — a TP shard
                                is then [Q_r; K_r; V_r], three row blocks stored one after the other.
                                With tp > n_kv_heads (KV-head replication, reading A30) the tp/n_kv_heads ranks of a KV
                                group each hold their share of the group's q heads and the WHOLE K and V head */
} etc_model_desc;

/* Megatron-style parallel configuration.  dist_opt = 1: MASTER/ADAM_M/ADAM_V are sharded over DP as
 * contiguous flat ranges of each (stage, tp-rank) local parameter space (reading A14); PARAM stays replicated.
 * pp_first / pp_last (f3, reading A27): number of layers on the first / last pipeline stage, 0 = not set (as
 * Megatron-LM's --decoder-first/last-pipeline-num-layers); the remaining layers are split evenly over the remaining
 * stages.  Both 0 = the even split the paper requires.
 * dist_opt_align (f3, reading A28): with dist_opt = 1 the DP shard size is rounded up to a multiple of this many
 * elements, chunk = ceil(Lloc / (dp*align)) * align (Megatron-LM pads its distributed-optimizer buffers so that every
 * DP shard is aligned); 0 or 1 = no rounding (reading A14); negative -> ETC_ERR_INVALID_ARG.  Padding is not stored:
 * a buffer holds only the real elements of its range.
 * vocab_divisor (f3, reading A31): > 0 pads the vocabulary dimension of word_embeddings / lm_head in this layout to
 * Vp = ceil(vocab / (vocab_divisor*tp)) * vocab_divisor*tp rows (Megatron-LM's --make-vocab-size-divisible-by, default
 * there 128); the padding rows [vocab, Vp) are stored in the shards like any other row.  0 = no padding, vocab % tp == 0
 * required (reading A12); negative -> ETC_ERR_INVALID_ARG.  Migration between layouts with different Vp: rows present on
 * both sides are moved (old padding rows included, so an identity reconfiguration is the identity), old rows beyond
 * the new Vp are dropped, new rows beyond the old Vp have no source and are ZERO-FILLED (`Fill`, next to the paper's
 * Send / Recv / Refer of PAPER.md:193-195); they count in need[] but in no traffic cell (etc_plan_stats.fill_bytes). */
typedef struct { int32_t tp, pp, dp, dist_opt, pp_first, pp_last, dist_opt_align, vocab_divisor; } etc_parallel_cfg;

typedef struct etc_layout etc_layout;   /* opaque, immutable after create */
typedef struct etc_plan etc_plan;       /* opaque, immutable after create */

/* Select the CUDA device the library works on (default 0).  Call once per process before anything else.  Calls that
 * create library-owned objects make that device current while they run and restore the caller's current device. */
etc_status etc_init(int32_t cuda_device);

/* (a1) Build the layout descriptor on the host and upload its piece tables.  *out is written only on success. */
etc_status etc_layout_create(const etc_model_desc* model, const etc_parallel_cfg* cfg, etc_layout** out);
void etc_layout_destroy(etc_layout* layout);
int32_t etc_layout_num_devices(const etc_layout* layout);                         /* tp*pp*dp */
int64_t etc_layout_num_pieces(const etc_layout* layout);                          /* index rectangles in the table */
/* bytes of the buffer of state kind `kind` (0..3) on device `dev`; 0 if the kind is absent; <0 on bad arguments */
int64_t etc_layout_buffer_bytes(const etc_layout* layout, int32_t dev, int32_t kind);

/* (a2) Cost matrix.  Device outputs, all int64:
 *   d_overlap [n_new][P] row-major: bytes held both by new rank n and by old device o (0 for o >= n_old)
 *   d_need    [n_new]: bytes new rank n needs;  d_hold [P]: bytes old device o holds (0 for o >= n_old)
 * Rows = curr ranks, columns = prev ranks, as in the paper (reading A1).  Enqueues on `stream`. */
etc_status etc_cost_matrix(const etc_layout* old_l, const etc_layout* new_l,
                           int64_t* d_overlap, int64_t* d_need, int64_t* d_hold, void* stream);

/* (a3) Migration sketch: device_map = argmax over injective maps pi:[0,n_new)->[0,P) of sum_n overlap[n][pi(n)]
 * (= Eq. 2's minimisation under Eq. 3/4, reading A4).  d_avail: optional device mask [P] (0 = device may not be
 * used, e.g. pre-empted; NULL = all usable).  method: ETC_SKETCH_HUNGARIAN = shortest augmenting paths (any P up to
 * ETC_SKETCH_MAX_P), ETC_SKETCH_EXHAUSTIVE = every injective map enumerated (P <= 8, the cross-check), ETC_SKETCH_AUTO
 * = the faster one (Hungarian).  For 32 < P <= 1024 the Hungarian method first tries the row-maximum certificate: if
 * every row can be given one of its maximal columns, that map attains the upper bound sum_n max_o overlap[n][o] and is
 * returned without a search (deterministic; the search runs otherwise, so the result is an optimum either way).
 * Outputs (device memory): d_device_map [n_new] int32, d_local_bytes [1] int64 = the achieved objective.  If no
 * feasible map exists both are filled with -1.  Enqueues on `stream`; no host synchronisation (a few KB of
 * stream-ordered scratch for P > 32). */
enum { ETC_SKETCH_AUTO = 0, ETC_SKETCH_EXHAUSTIVE = 1, ETC_SKETCH_HUNGARIAN = 2 };
etc_status etc_sketch(const int64_t* d_overlap, int32_t n_new, int32_t P, const uint8_t* d_avail, int32_t method,
                      int32_t* d_device_map, int64_t* d_local_bytes, void* stream);

/* (a3) The same sketch for callers that cannot allocate device memory.  etc_sketch takes a few KB of work area from
 * CUDA's stream-ordered pool whenever P > 32.  Three kinds of caller cannot afford that:
 *   - a trainer whose own caching allocator has already claimed all free HBM (the migration runs exactly when the GPU is
 *     at its fullest: old state, new state and staging together, 136 of 180 GB on the largest benchmark config), so a
 *     driver-level allocation made behind its back fails with out-of-memory, or forces it to give memory back;
 *   - a failure-recovery handler that must not stall: growing a memory pool, like cudaMalloc / cudaFree, may wait for
 *     every stream of the device, including the ones still running the surviving ranks' work;
 *   - a process that was given a fixed device-memory budget up front and is not allowed to exceed it later.
 * etc_sketch_static computes what etc_sketch(..., ETC_SKETCH_HUNGARIAN, ...) computes — same arguments (minus `method`),
 * same outputs, the same device_map bit for bit (warp search for P <= 32; row-maximum certificate, then the CTA search,
 * for P > 32) — and calls no cudaMalloc, cudaMallocAsync, cudaFree or any library routine that allocates.  Its work area is
 * a fixed array of ETC_SKETCH_STATIC_SCRATCH_BYTES (28 KB) inside libetc.so's device image: every GPU that loads the
 * library holds those 28 KB until the process exits, whether or not this entry point is ever called.
 * Limit: P <= ETC_SKETCH_STATIC_MAX_P (1024 devices; the paper's Algorithm 1 is quoted for k < 1024).  A
 * larger P is refused with ETC_ERR_WORKSPACE and a text in etc_last_error_detail(); nothing is launched or written.
 * Rules that come with a shared, resident work area:
 *   - The first call on a device looks up where the array lives on that device (cudaGetSymbolAddress, which may also make
 *     the CUDA runtime load the library's kernels).  Make that first call during start-up, outside any stream capture and
 *     outside the time-critical path; later calls on the device only launch kernels.
 *   - All calls share the one array, and it keeps what the previous call wrote.  No part of it needs clearing: each call
 *     overwrites every entry it later reads.  But two calls whose kernels can run at the same time on one GPU (different
 *     streams without an ordering between them, or two host threads doing that) overwrite each other's rows and the
 *     results are undefined: keep calls on one stream, or order them with events.  Calls on different GPUs do not
 *     interact (each device has its own copy of the array).
 *   - The caller still owns and passes d_overlap, d_avail, d_device_map and d_local_bytes as for etc_sketch; if no
 *     feasible map exists both outputs are filled with -1.  Enqueues on `stream`; no host synchronisation. */
#define ETC_SKETCH_STATIC_MAX_P 1024
#define ETC_SKETCH_STATIC_SCRATCH_BYTES 28672
etc_status etc_sketch_static(const int64_t* d_overlap, int32_t n_new, int32_t P, const uint8_t* d_avail,
                             int32_t* d_device_map, int64_t* d_local_bytes, void* stream);

/* (f1) Virtual rank allocator: Algorithm 2 "Placement-Aware Remapping" (the garbled listing is read
 * from the prose PAPER.md:220-222, reading A23) composed with the sketch into one final device map
 * (communication coalescing): pass d_out_map to etc_plan_create and every element moves in ONE hop.
 *   d_device_map [cw] int32 (device memory): the sketch, curr rank -> physical device, injective into [0,P),
 *                 P = max(pw, cw); pw / cw = world size of the prev / curr state; devices_per_node = n of Algorithm 2.
 *   mode: ETC_DEFRAG_OCCUPANCY (lines 1-9: idle devices in ascending order are paired with occupied devices in descending
 *         order until they meet, so the occupied devices become exactly [0,cw) and whole nodes are freed),
 *         ETC_DEFRAG_EFFICIENCY (lines 10-20: every device of a fragmented node takes its target rank, rank k on device k,
 *         so each TP group sits inside a node; the target placement is fixed by the rank order alone, so this stage
 *         OVERRIDES the sketch on every fragmented node — on its own it returns the identity placement wherever the
 *         sketch differs from it — and `pw` only bounds the device ids accepted in d_device_map),
 *         ETC_DEFRAG_BOTH (occupancy, then efficiency on its result).
 * Outputs (device memory): d_out_map [cw] int32 (must not alias d_device_map); d_n_ops [2] int32 = number of migration
 * operators of the occupancy and of the efficiency stage; d_ops: optional (NULL to skip) [2][cw][2] int32, operators
 * <a,b> in the paper's order: occupancy <idle device, occupied device> at d_ops[0..], efficiency <target rank, current
 * load or -1> at d_ops[2*cw..].  If the input is not an injective map, d_out_map is filled with -1 and d_n_ops with -1.
 * Enqueues on `stream`; no host synchronisation. */
enum { ETC_DEFRAG_OCCUPANCY = 1, ETC_DEFRAG_EFFICIENCY = 2, ETC_DEFRAG_BOTH = 3 };
etc_status etc_defrag(const int32_t* d_device_map, int32_t pw, int32_t cw, int32_t devices_per_node, int32_t mode,
                      int32_t* d_out_map, int32_t* d_ops, int32_t* d_n_ops, void* stream);

/* (a4) Plan.  device_map: [n_new] int32, host OR device pointer.  flags: ETC_LOCAL_DIRECT (slices whose source device
 * is the destination device are copied old buffer -> new buffer, never staged: the paper's Refer, reading A19) or
 * ETC_ALL_STAGED (every slice goes through pack/unpack: a measurement mode); OR-ed with ETC_KIND_MAJOR to order
 * slices, chunks and staging segments by state kind first (one segment per (kind, source, destination) instead of one
 * per (source, destination)): required for state chunking, etc_plan_set_rounds below.  ETC_ALL_DIRECT (not with
 * ETC_ALL_STAGED): NO slice is staged, every one is copied source buffer -> destination buffer in one hop — for shards
 * that all live in one address space anyway (pinned host memory: the zero-copy pipeline), where a staging buffer
 * stands for no message; the traffic matrix and remote_bytes are unchanged, staging_bytes = 0.  Synchronises `stream` once
 * (sizes must come back to the host) and then enqueues the kernels that write the slice and chunk tables: the plan is
 * complete in `stream` order, not on return.  Every later call that reads the plan on ANOTHER stream (etc_migrate*,
 * etc_plan_set_rounds, etc_plan_validate) makes that stream wait for those kernels itself (an event recorded at the end
 * of this call), so no caller-side ordering is needed.  Fails with ETC_ERR_BAD_MAP if the map is not injective into
 * [0,P). */
enum { ETC_LOCAL_DIRECT = 0, ETC_ALL_STAGED = 1, ETC_KIND_MAJOR = 2, ETC_ALL_DIRECT = 4, ETC_NO_SYNC = 8, ETC_NO_REORDER = 16 };
/* ETC_NO_SYNC (OR-ed into flags): etc_plan_create does NOT synchronise.  The slice / chunk tables are sized from upper
 * bounds the host derives from the two layouts (pieces per tensor, bytes needed), the real counts stay on the device, and
 * etc_migrate / etc_migrate_phase launch bound-sized grids whose surplus CTAs leave at once: a whole reconfiguration is
 * then one uninterrupted submission (etc_migrate_state below).  The staging buffer must hold etc_staging_bound() bytes
 * (the exact size is not known to the host).  A bad device map, an unrecoverable failure mask or (never observed) a
 * bound that falls short is detected ON THE DEVICE: the plan then copies nothing, and the error is reported by the
 * first call that needs the counts on the host — etc_plan_get_stats (which waits for the plan's kernels), and likewise
 * etc_plan_get_traffic / _slices / _fills / etc_plan_set_rounds / etc_plan_validate.  A hint: plans whose bound exceeds
 * 32 768 copy work items (states beyond ~1 GB) are made the synchronising way — their copy kernels dwarf one host sync,
 * and the surplus CTAs of a bound-sized grid would cost more than it.
 * Launch order.  A plan also keeps its copy
 * work items in ADDRESS order — launch 1 (pack + local) by source address, launch 2 (unpack) by destination address —
 * and etc_migrate / etc_migrate_phase walk those lists: work items that read interleaved column blocks of the same
 * rows (a TP change of a row-parallel weight), or the same source range for several new ranks (replicated state fanning
 * out to more DP groups), then run side by side and share DRAM pages and L2 lines.  The result is the same bytes either
 * way.  etc_plan_set_rounds builds the same lists per round, so etc_migrate_round walks each round in address order too.
 * A bound-sized ETC_NO_SYNC plan keeps the lists if its state exceeds 128 MB (about the L2: below that the order is
 * moot).  ETC_NO_REORDER (OR-ed into flags) keeps every launch in list order (unit by unit): a measurement mode. */
int64_t etc_staging_bound(const etc_layout* old_l, const etc_layout* new_l, int32_t flags);   /* bytes; < 0 on bad arguments */
etc_status etc_plan_create(const etc_layout* old_l, const etc_layout* new_l, const int32_t* device_map,
                           int32_t flags, etc_plan** out, void* stream);
/* Whether ETC_NO_SYNC was honoured for this plan: 1 = deferred (tables sized from host-side bounds, counts still on the
 * device, etc_plan_create did not synchronise — safe inside a stream capture), 0 = made the synchronising way (no
 * ETC_NO_SYNC flag, or the bound exceeded 32 768 copy work items: etc_plan_create called cudaStreamSynchronize, which is
 * not allowed while `stream` is being captured — probe with a plan made outside the capture first), < 0 on a NULL plan.
 * Host-only; never synchronises. */
int32_t etc_plan_is_deferred(const etc_plan* plan);
/* Releases the plan's tables in stream order, behind everything already enqueued that reads them (on whatever streams):
 * safe to call right after the last etc_migrate* call on the plan, while its kernels are still queued.  Do call it there
 * when migrations are pipelined: the tables return to the stream-ordered pool at that point of the copy stream, and a plan
 * dropped a step later is only reusable a step later (bench.py keeps three steps in flight and releases each plan right
 * behind its own launches). */
void etc_plan_destroy(etc_plan* plan);

/* (f4) Failure-aware sourcing ("Fault-tolerance through DP": "the workload on the failed device can be
 * obtained from other DP groups via the PP/TP ranks"; reading A26).  failed: [n_old] uint8, host OR device
 * pointer, nonzero = old device lost with everything it held (NULL = no failures = etc_plan_create).  A failed device is
 * never a source (not even a local one: its physical slot may host a new rank, which then receives everything); where
 * the designated holder (d,s,r) of reading A6 failed, the source is the next surviving DP replica (d+1, d+2, ... mod
 * dp_old, same s and r).  With dp_old = d this survives any d-1 failures.  ETC_ERR_UNRECOVERABLE if some needed element
 * has no surviving holder (all replicas failed, or a DP-sharded distributed-optimizer range whose only holder failed).
 * etc_mask_failed zeroes the failed devices' columns of d_overlap [n_new][P] and entries of d_hold [P] (may be NULL),
 * so that etc_sketch counts nothing as local on them; d_failed is a DEVICE pointer [n_old].  Enqueues on `stream`. */
etc_status etc_plan_create_failed(const etc_layout* old_l, const etc_layout* new_l, const int32_t* device_map,
                                  const uint8_t* failed, int32_t flags, etc_plan** out, void* stream);
etc_status etc_mask_failed(int64_t* d_overlap, int64_t* d_hold, int32_t n_new, int32_t n_old, int32_t P,
                           const uint8_t* d_failed, void* stream);

/* The paper's own treatment of the DP dimension ("we isolate the PP/TP processes under different DP
 * ranks ... the difference between the workloads to be infinite"; reading A5 explains why the default matrix
 * spans all DP x PP x TP devices instead): zero, in place, every cell of d_overlap [n_new][P] whose new rank and old
 * device have different DP ranks, so that etc_sketch keeps no bytes local across DP groups.  Enqueues on `stream`. */
etc_status etc_mask_cross_dp(const etc_layout* old_l, const etc_layout* new_l, int64_t* d_overlap, void* stream);

typedef struct {
  int64_t staging_bytes;   /* size the caller must allocate for `staging` (payload + alignment padding) */
  int64_t local_bytes;     /* payload bytes whose source device is their destination device */
  int64_t remote_bytes;    /* payload bytes that change device (sum of off-diagonal traffic) */
  int64_t staged_bytes;    /* payload bytes that go through pack/unpack (= remote_bytes, or all bytes if ALL_STAGED) */
  int64_t n_slices_local, n_slices_staged;   /* 2-D strided copy descriptors */
  int64_t n_chunks_local, n_chunks_staged;   /* copy work items (<= ETC_CHUNK_BYTES each) */
  int32_t n_old, n_new, P, flags;
  int64_t fill_bytes;      /* destination bytes with no source, zero-filled (grown padded vocabulary, reading A31);
                              local_bytes + remote_bytes + fill_bytes = sum of need[] */
  int64_t n_fills;         /* zero-fill descriptors */
} etc_plan_stats;
etc_status etc_plan_get_stats(const etc_plan* plan, etc_plan_stats* out);
/* traffic matrix T [P][P] row-major, int64, copied to HOST memory: T[o][p] = payload bytes whose source is old device
 * o and whose destination is physical device p (diagonal = local bytes).  Synchronous. */
etc_status etc_plan_get_traffic(const etc_plan* plan, int64_t* h_traffic);

/* The device map the plan was made for, [n_new] int32 copied to HOST memory (e.g. the sketch etc_migrate_state chose).
 * Synchronous. */
etc_status etc_plan_get_map(const etc_plan* plan, int32_t* h_device_map);

/* One slice = one 2-D strided copy (rows x row_bytes).  For tests / inspection; copied to HOST memory.
 * which = 0: staged slices, 1: local slices.  h_out must hold n_slices_* entries. */
typedef struct {
  int64_t src_off, dst_off, stg_off;          /* byte offsets inside src buffer, dst buffer, staging buffer (-1: none) */
  int64_t row_bytes;                          /* contiguous bytes per row */
  int32_t src_stride, dst_stride;             /* row pitch in bytes on each side (in staging the pitch is row_bytes) */
  int32_t nrows;
  int32_t src_dev, dst_rank, dst_phys, kind;  /* src buffer = src_bufs[src_dev*4+kind], dst = dst_bufs[dst_rank*4+kind] */
  int32_t pad;
} etc_slice;
etc_status etc_plan_get_slices(const etc_plan* plan, int32_t which, etc_slice* h_out);
/* The copy work items ("chunks": at most ETC_CHUNK_BYTES of payload each, nrows x row_bytes with a row pitch per side;
 * what one CTA of the copy kernels moves).  which = 0: the staged chunks in plan order (unit by unit), 1: the local
 * chunks in plan order, 2: the launch-1 list in address order (every chunk of pack + local sorted by source address;
 * `staged` tells the two apart), 3: the launch-2 list (the staged chunks sorted by destination address).  h_out must
 * hold n_chunks_staged (0, 3), n_chunks_local (1) or their sum (2) entries; copied to HOST memory.  2 and 3 return
 * ETC_ERR_INVALID_ARG for a plan that keeps no ordered lists (ETC_NO_REORDER, or a bound-sized ETC_NO_SYNC plan of a
 * state below 128 MB).
 * Address order means: non-decreasing buffer index, and inside a buffer non-decreasing 64 KB block of the offset (for
 * layouts beyond 256 GB in all, a coarser block); the order inside a block is unspecified. */
typedef struct {
  int64_t src_off, dst_off, stg_off;  /* byte offsets in the source buffer, destination buffer, staging buffer */
  int32_t src_stride, dst_stride;     /* row pitch in bytes (the staging pitch is row_bytes) */
  int32_t row_bytes, nrows;
  uint16_t src_buf, dst_buf;          /* old_dev*4+kind, new_rank*4+kind */
  int16_t vec;                        /* widest power-of-two access (<= 16 B) every address of the chunk is aligned to */
  int16_t staged;                     /* lists 2: 1 = packed into staging, 0 = copied old -> new buffer; else 0 */
} etc_chunk;
etc_status etc_plan_get_chunks(const etc_plan* plan, int32_t which, etc_chunk* h_out);
/* Bounds check of a finished plan, on the device: counts the copy work items whose source, destination or staging
 * extent does not lie inside the buffer it addresses (sizes from the layouts the plan was made from), or whose declared
 * access width does not divide its addresses; the address-ordered launch lists (whole-plan and per-round) are checked
 * the same way and must be permutations of the plan's lists (order-independent checksums), else one more is counted.
 * *n_bad (HOST) = 0 for every plan this library makes; a debugging and test aid (one thread per work item,
 * synchronises `stream`). */
etc_status etc_plan_validate(const etc_plan* plan, int64_t* n_bad, void* stream);
/* The zero-fill descriptors (reading A31) as etc_slice records with no source: src_dev = -1, src_off = stg_off = -1,
 * src_stride = 0; h_out must hold etc_plan_stats.n_fills entries (order unspecified).  Copied to HOST memory. */
etc_status etc_plan_get_fills(const etc_plan* plan, etc_slice* h_out);

/* (a5,a6) Migrate.  src_bufs[old_dev*4 + kind], dst_bufs[new_rank*4 + kind]: HOST arrays of DEVICE pointers (NULL
 * where the buffer has 0 bytes), each 16-byte aligned and at least etc_layout_buffer_bytes() long.  A buffer may also
 * live in PINNED HOST memory (cudaMallocHost / cudaHostAlloc: device-addressable at the same address): the copy kernels
 * then read or write it over PCIe themselves ("zero-copy"), touching only the bytes their chunks name, and no device
 * copy of that shard is needed.  staging: device
 * pointer, >= staging_bytes (may be NULL if staging_bytes == 0).  Enqueues on `stream`:
 *   ETC_PHASE_PACK   : pack staged slices old buffers -> staging, copy local slices old -> new directly, and zero-fill
 *                      the destination bytes that have no source (reading A31; none unless the padded vocabulary grew)
 *   ETC_PHASE_UNPACK : unpack staged slices staging -> new buffers
 * etc_migrate runs both phases.  No allocation, no host synchronisation.  Every destination byte is written exactly
 * once.  Concurrency: a plan is immutable and may be used by several etc_migrate* calls at once, from different host
 * threads and on different streams, each with its own buffer set (double-buffered payloads, a captured CUDA graph
 * replayed beside a live call): with (n_old + n_new) <= 96 the pointer tables travel in each launch's kernel
 * parameters.  Beyond 96 devices the tables are written into one device table per plan (per round for
 * etc_migrate_round) by a kernel on `stream`: such calls on the SAME plan must then be ordered one after the other (same
 * stream, or events) unless they pass identical buffer sets. */
enum { ETC_PHASE_PACK = 1, ETC_PHASE_UNPACK = 2, ETC_PHASE_ALL = 3 };
etc_status etc_migrate(const etc_plan* plan, const void* const* src_bufs, void* const* dst_bufs,
                       void* staging, void* stream);
etc_status etc_migrate_phase(const etc_plan* plan, const void* const* src_bufs, void* const* dst_bufs,
                             void* staging, int32_t phases, void* stream);

/* The migration primitive in ONE call (previous configuration, current configuration, model state
 * in; migrated state out): (a1) both layout descriptors, (a2) cost matrix, (a3) sketch (d_avail: optional device mask
 * [P], as etc_sketch), (a4) plan with ETC_NO_SYNC, (a5, a6) pack / unpack / local — enqueued back to back on `stream`
 * without any host synchronisation; returns as soon as everything is enqueued.  staging / staging_bytes: device buffer
 * of at least etc_staging_bound() bytes for these two layouts (ETC_ERR_WORKSPACE if smaller; may be NULL / 0 with
 * ETC_ALL_DIRECT).  flags: ETC_LOCAL_DIRECT | ETC_ALL_STAGED | ETC_ALL_DIRECT.  plan_out: optional; receives the plan
 * (caller destroys it) so that the chosen map's statistics and any device-side error can be read with
 * etc_plan_get_stats afterwards; with NULL a device-side error (e.g. no feasible sketch under d_avail) leaves the
 * destination buffers unwritten and goes unreported. */
etc_status etc_migrate_state(const etc_model_desc* model, const etc_parallel_cfg* old_cfg, const etc_parallel_cfg* new_cfg,
                             const void* const* src_bufs, void* const* dst_bufs, void* staging, int64_t staging_bytes,
                             const uint8_t* d_avail, int32_t flags, etc_plan** plan_out, void* stream);

#define ETC_CHUNK_BYTES 65536

/* (f2) State chunking with bounded staging and eager release ("state chunking to migrate states in
 * sequential chunks with on-demand buffer allocation, and eager release of source-side state ... after each round";
 * :378 "reduces the peak to one optimizer component at a time").  For a plan created with ETC_KIND_MAJOR,
 * etc_plan_set_rounds cuts the migration into rounds, kind by kind (PARAM, MASTER, ADAM_M, ADAM_V), each kind into as
 * many rounds as it takes for every round to use at most max_staging_bytes (>= 2*ETC_CHUNK_BYTES) of staging.
 * Synchronises `stream` once (round sizes come back to the host).  May be called again with another bound.
 * etc_migrate_round enqueues round `round` (pack + local, unpack; `phases` as in etc_migrate_phase).  It reads only the
 * source buffers and writes only the destination buffers of the round's kind (the kind's zero-fills, reading A31, go
 * with its first round): pointers of other kinds are not looked
 * at (they may be NULL: already released, or not yet allocated).  `staging` needs only etc_round_info.staging_bytes
 * bytes and may be reused by the next round on the same stream.  After all rounds every destination byte has been
 * written exactly once, bit-identical to etc_migrate. */
typedef struct {
  int32_t kind, sub, n_sub, pad;     /* state kind; round `sub` of `n_sub` of that kind */
  int64_t staging_bytes;             /* staging bytes this round uses (<= max_staging_bytes) */
  int64_t staged_bytes, local_bytes; /* payload bytes through pack/unpack, and copied directly */
  int64_t n_chunks_staged, n_chunks_local;
} etc_round_info;
etc_status etc_plan_set_rounds(etc_plan* plan, int64_t max_staging_bytes, int32_t* n_rounds, void* stream);
etc_status etc_plan_get_round(const etc_plan* plan, int32_t round, etc_round_info* out);
etc_status etc_migrate_round(const etc_plan* plan, int32_t round, const void* const* src_bufs, void* const* dst_bufs,
                             void* staging, int32_t phases, void* stream);

/* Host-resident old shards: upload exactly the source bytes the plan reads (only the slices named by
 * the migration instructions move).  h_src_bufs / d_src_bufs: HOST arrays [n_old*4] of pointers to the host copy
 * (pinned memory, or the copies are not asynchronous) and the device copy of each old shard buffer; every region a
 * slice of the plan reads (rows x row_bytes at the buffer's pitch) is copied from the host buffer to the same offset
 * of the device buffer with cudaMemcpyAsync / cudaMemcpy2DAsync on `stream`; regions read by several slices are
 * copied once; bytes no slice reads are not transferred and stay undefined on the device (etc_migrate never reads
 * them).  only_kind = 0..3 restricts the call to one state kind (pipelining with rounds), -1 = all kinds.
 * *bytes_out (optional) receives the bytes enqueued.  The first call on a plan synchronises the stream the plan was
 * created on (the slice table comes back to the host once). */
etc_status etc_upload_sources(const etc_plan* plan, const void* const* h_src_bufs, void* const* d_src_bufs,
                              int32_t only_kind, int64_t* bytes_out, void* stream);

const char* etc_status_string(etc_status s);   /* static strings */
const char* etc_last_error_detail(void);       /* thread-local; CUDA error text after ETC_ERR_CUDA, else "" */
int64_t etc_kernel_launches(void);             /* number of kernels this library has launched in this process */

#ifdef __cplusplus
}
#endif
#endif /* ETC_H_ */
