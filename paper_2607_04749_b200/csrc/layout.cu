// layout.cu — (a1) layout descriptor: (model_desc, parallel_cfg) -> index rectangles ("pieces") of every state tensor
// on every device, uploaded once.  Host-side integer bookkeeping only (PAPER.md:106 workload abstraction; :110 "each
// device can derive its workload following these rules"; :199 TP slices -> explicit split types, reading A8).
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>
#include "etc_internal.h"

namespace etc {

static thread_local std::string g_detail;
static int g_device = 0;
static long long g_launches = 0;

void set_error_detail(const char* what, cudaError_t e) {
  g_detail = std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
  (void)cudaGetLastError();
}
void set_error_text(const char* text) { g_detail = text; }
void clear_error_detail() { g_detail.clear(); }
void count_launch(int n) { __atomic_add_fetch(&g_launches, (long long)n, __ATOMIC_RELAXED); }
int current_device() { return g_device; }

struct LTensor { int64_t rows, cols; int32_t split, where, layer; };   // where: 0 pre, 1 layer, 2 post

// Logical tensor list in id order.  The fused QKV weight / bias has its own split type
// (readings A10, A29, A30: row order and KV-head replication, see qkv_blocks); SwiGLU fc1 = [gate; up] is COL2.
// rows of the embedding tensors: the vocabulary padded to a multiple of vocab_divisor * tp (reading A31)
static int64_t vocab_rows(const etc_model_desc& m, const etc_parallel_cfg& c) {
  if (c.vocab_divisor <= 0) return m.vocab;
  const int64_t unit = (int64_t)c.vocab_divisor * c.tp;
  return ((int64_t)m.vocab + unit - 1) / unit * unit;
}

static std::vector<LTensor> logical_tensors(const etc_model_desc& m, const etc_parallel_cfg& c) {
  std::vector<LTensor> v;
  const int64_t V = vocab_rows(m, c);
  const int64_t h = m.hidden, d = m.head_dim, f = m.ffn_hidden;
  const int64_t qkv = (int64_t(m.n_q_heads) + 2 * int64_t(m.n_kv_heads)) * d, qd = int64_t(m.n_q_heads) * d;
  v.push_back({V, h, COL, 0, -1});
  if (m.style == ETC_GPT && m.max_pos > 0) v.push_back({m.max_pos, h, REPL, 0, -1});
  for (int l = 0; l < m.n_layers; ++l) {
    if (m.style == ETC_GPT) {
      v.push_back({1, h, REPL, 1, l}); v.push_back({1, h, REPL, 1, l});          // ln1 w,b
      v.push_back({qkv, h, QKV, 1, l}); v.push_back({qkv, 1, QKV, 1, l});        // qkv w,b
      v.push_back({h, qd, ROW, 1, l}); v.push_back({1, h, REPL, 1, l});          // proj w,b
      v.push_back({1, h, REPL, 1, l}); v.push_back({1, h, REPL, 1, l});          // ln2 w,b
      v.push_back({f, h, COL, 1, l}); v.push_back({f, 1, COL, 1, l});            // fc1 w,b
      v.push_back({h, f, ROW, 1, l}); v.push_back({1, h, REPL, 1, l});           // fc2 w,b
    } else {
      v.push_back({1, h, REPL, 1, l});                                           // ln1 w
      v.push_back({qkv, h, QKV, 1, l});                                          // qkv w
      v.push_back({h, qd, ROW, 1, l});                                           // proj w
      v.push_back({1, h, REPL, 1, l});                                           // ln2 w
      v.push_back({2 * f, h, COL2, 1, l});                                       // fc1 w = [gate; up]
      v.push_back({h, f, ROW, 1, l});                                            // fc2 w
    }
  }
  v.push_back({1, h, REPL, 2, -1});                                              // final_ln w
  if (m.style == ETC_GPT) v.push_back({1, h, REPL, 2, -1});                      // final_ln b
  if (!m.tied_embeddings) v.push_back({V, h, COL, 2, -1});                       // lm_head
  return v;
}

// First layer of pipeline stage s (s = pp -> n_layers); even split unless pp_first / pp_last are set (reading A27).
// -1: impossible split, -2: invalid arguments.
static int stage_begin(int n_layers, const etc_parallel_cfg& c, int s) {
  if (c.pp_first < 0 || c.pp_last < 0 || ((c.pp_first || c.pp_last) && c.pp < 2)) return -2;
  const int fixed_stages = (c.pp_first ? 1 : 0) + (c.pp_last ? 1 : 0);
  const int free_stages = c.pp - fixed_stages, free_layers = n_layers - c.pp_first - c.pp_last;
  if (free_stages < 0 || free_layers < 0) return -1;
  if (free_stages == 0 ? free_layers != 0 : (free_layers % free_stages != 0 || free_layers < free_stages)) return -1;
  const int per = free_stages ? free_layers / free_stages : 0;
  if (s <= 0) return 0;
  if (s >= c.pp) return n_layers;
  return c.pp_first ? c.pp_first + (s - 1) * per : s * per;
}

etc_status validate_config(const etc_model_desc* m, const etc_parallel_cfg* c) {
  if (!m || !c) return ETC_ERR_INVALID_ARG;
  if (c->tp < 1 || c->pp < 1 || c->dp < 1 || (c->dist_opt != 0 && c->dist_opt != 1) || c->dist_opt_align < 0 ||
      c->vocab_divisor < 0) return ETC_ERR_INVALID_ARG;
  if (m->style != ETC_GPT && m->style != ETC_LLAMA) return ETC_ERR_INVALID_ARG;
  if (m->n_layers < 1 || m->hidden < 1 || m->n_q_heads < 1 || m->n_kv_heads < 1 || m->head_dim < 1 ||
      m->ffn_hidden < 1 || m->vocab < 1 || m->max_pos < 0) return ETC_ERR_INVALID_ARG;
  if (m->param_dtype != ETC_BF16 && m->param_dtype != ETC_FP32) return ETC_ERR_INVALID_ARG;
  if (m->kinds <= 0 || m->kinds > 15) return ETC_ERR_INVALID_ARG;
  if (m->tied_embeddings != 0 && m->tied_embeddings != 1) return ETC_ERR_INVALID_ARG;
  if (m->n_q_heads % m->n_kv_heads) return ETC_ERR_INVALID_ARG;
  if (int64_t(c->tp) * c->pp * c->dp > 32767) return ETC_ERR_INVALID_ARG;
  if (m->qkv_order != ETC_QKV_GROUPED && m->qkv_order != ETC_QKV_BLOCKED) return ETC_ERR_INVALID_ARG;
  if (c->tp > m->n_kv_heads) {                               // KV-head replication (reading A30)
    const int rep = c->tp / m->n_kv_heads;
    if (c->tp % m->n_kv_heads || (m->n_q_heads / m->n_kv_heads) % rep) return ETC_ERR_UNSUPPORTED;
  }
  { const int sb = stage_begin(m->n_layers, *c, 0); if (sb < 0) return sb == -2 ? ETC_ERR_INVALID_ARG : ETC_ERR_INDIVISIBLE; }
  if ((c->tp <= m->n_kv_heads && m->n_kv_heads % c->tp) || m->ffn_hidden % c->tp ||
      (c->vocab_divisor == 0 && m->vocab % c->tp)) return ETC_ERR_INDIVISIBLE;
  return ETC_OK;
}

}  // namespace etc

using namespace etc;

extern "C" etc_status etc_init(int32_t cuda_device) {
  clear_error_detail();
  int n = 0;
  ETC_CUDA_TRY(cudaGetDeviceCount(&n));
  if (cuda_device < 0 || cuda_device >= n) return ETC_ERR_INVALID_ARG;
  ETC_CUDA_TRY(cudaSetDevice(cuda_device));
  g_device = cuda_device;
  // keep stream-ordered allocations cached: plan creation allocates and frees tables on every call
  cudaMemPool_t pool;
  ETC_CUDA_TRY(cudaDeviceGetDefaultMemPool(&pool, cuda_device));
  uint64_t thr = UINT64_MAX;
  ETC_CUDA_TRY(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr));
  return ETC_OK;
}

// Pinned slabs + private upload stream: the layout tables are built straight into a pinned slab and uploaded with one
// async copy on the upload stream.  etc_layout_create does not wait for the copy: it records the layout's `ready` event
// behind it, and every call that reads the tables on a stream makes that stream wait for the event (layout_use).  A slab
// is reused only after the upload that last read it has finished (its `done` event; with N_SLABS uploads in flight this
// wait is never taken in practice).
namespace etc {
static std::mutex g_up_mu;
static cudaStream_t g_up_stream = nullptr;
constexpr int N_SLABS = 8;
struct Slab { void* p = nullptr; size_t cap = 0; cudaEvent_t done = nullptr; bool in_flight = false; bool busy = false; };
static Slab g_slabs[N_SLABS];
static unsigned g_slab_next = 0;
static cudaError_t slab_acquire(size_t bytes, Slab** out) {
  if (!g_up_stream) { cudaError_t e = cudaStreamCreateWithFlags(&g_up_stream, cudaStreamNonBlocking); if (e) return e; }
  // the next slab that no other host thread is building a layout in (two builders at most in this library: primitive.cu)
  Slab* pick = nullptr;
  for (int t = 0; t < N_SLABS && !pick; ++t) { Slab& c = g_slabs[g_slab_next++ % N_SLABS]; if (!c.busy) pick = &c; }
  if (!pick) return cudaErrorNotReady;
  Slab& s = *pick;
  if (!s.done) { cudaError_t e = cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming); if (e) return e; }
  if (s.in_flight) { cudaError_t e = cudaEventSynchronize(s.done); if (e) return e; s.in_flight = false; }
  if (bytes > s.cap) {
    if (s.p) cudaFreeHost(s.p);
    s.p = nullptr; s.cap = 0;
    const size_t cap = std::max<size_t>(bytes + bytes / 2, 1 << 20);
    cudaError_t e = cudaMallocHost(&s.p, cap); if (e) return e;
    s.cap = cap;
  }
  s.busy = true;                                         // until the upload has been enqueued (etc_layout_create)
  *out = &s;
  return cudaSuccess;
}

// Call before enqueueing anything that reads the layout's device tables on `st`.
cudaError_t layout_use(const etc_layout* L, cudaStream_t st) {
  cudaError_t e = cudaSuccess;
  if (L->ready) {
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    e = cudaStreamIsCapturing(st, &cap);
    if (e == cudaSuccess)
      e = cudaStreamWaitEvent(st, L->ready, cap == cudaStreamCaptureStatusActive ? cudaEventWaitExternal : cudaEventWaitDefault);
  }
  L->streams.note(st);
  return e;
}
// TP shard of one tensor instance: up to 3 row blocks (first logical row rb, rows nr, first local row ls) stored one
// after the other, times a column range.  rep / rbase per block: the TP ranks [rbase, rbase + rep) hold its elements.
struct Sh { int64_t start, n, rb[3], nr[3], ls[3], c0, W; int nblk; int16_t rep[3], rbase[3]; int32_t lt; uint16_t flags; };

// Row blocks of the fused QKV tensor on TP rank r (q = n_q heads, k = n_kv heads, d rows per head, qpg = q/k):
//   tp <= k: the rank holds kpr = k/tp whole KV groups.  GROUPED order: they are one contiguous row range (reading
//            A10).  BLOCKED order ([Q;K;V], reading A29): [Q_r; K_r; V_r], three blocks.
//   tp >  k: rep = tp/k ranks share KV group g = r/rep (reading A30); rank r holds the (r % rep)-th share of the group's
//            q heads and the whole K and V head of the group, which are therefore held by rep ranks.
static void qkv_blocks(const etc_model_desc& m, int tp, int r, Sh& s) {
  const int64_t q = m.n_q_heads, k = m.n_kv_heads, d = m.head_dim, qpg = q / k;
  if (tp <= k) {
    const int64_t kpr = k / tp;
    if (m.qkv_order == ETC_QKV_GROUPED) { s.nr[0] = kpr * (qpg + 2) * d; s.rb[0] = r * s.nr[0]; return; }
    s.nblk = 3;
    s.nr[0] = q / tp * d; s.rb[0] = r * s.nr[0];
    s.nr[1] = s.nr[2] = kpr * d; s.rb[1] = q * d + r * kpr * d; s.rb[2] = (q + k) * d + r * kpr * d;
    return;
  }
  const int64_t rep = tp / k, g = r / rep, share = r % rep, qpr = qpg / rep;
  if (m.qkv_order == ETC_QKV_GROUPED) {
    const int64_t g0 = g * (qpg + 2) * d;
    s.nblk = 2;
    s.nr[0] = qpr * d; s.rb[0] = g0 + share * qpr * d;
    s.nr[1] = 2 * d;   s.rb[1] = g0 + qpg * d;
    s.rep[1] = (int16_t)rep; s.rbase[1] = (int16_t)(g * rep);
  } else {
    s.nblk = 3;
    s.nr[0] = qpr * d; s.rb[0] = r * qpr * d;
    s.nr[1] = s.nr[2] = d; s.rb[1] = q * d + g * d; s.rb[2] = (q + k) * d + g * d;
    s.rep[1] = s.rep[2] = (int16_t)rep; s.rbase[1] = s.rbase[2] = (int16_t)(g * rep);
  }
}
}  // namespace etc

extern "C" etc_status etc_layout_create(const etc_model_desc* model, const etc_parallel_cfg* cfg, etc_layout** out) {
  clear_error_detail();
  if (!out) return ETC_ERR_INVALID_ARG;
  etc_status st = validate_config(model, cfg);
  if (st != ETC_OK) return st;
  const etc_model_desc& m = *model;
  const int tp = cfg->tp, pp = cfg->pp, dp = cfg->dp;
  const int n_dev = tp * pp * dp;
  const std::vector<LTensor> lts = logical_tensors(m, *cfg);
  if (vocab_rows(m, *cfg) > INT32_MAX) return ETC_ERR_INVALID_ARG;
  const int nT = (int)lts.size(), nG = nT * ETC_NUM_KINDS;
  int max_stage_layers = 0;
  for (int s = 0; s < pp; ++s) max_stage_layers = std::max(max_stage_layers, stage_begin(m.n_layers, *cfg, s + 1) - stage_begin(m.n_layers, *cfg, s));
  const bool two_inst = m.tied_embeddings && pp > 1;     // word_embeddings held by first AND last stage
  const int mask_words = (nT + 31) / 32;
  int n_kinds = 0; for (int k = 0; k < ETC_NUM_KINDS; ++k) n_kinds += (m.kinds >> k) & 1;

  // blob: dev_start | first | ltmask | kind_start | pieces (pieces last: their count is known only after the build)
  auto al = [](size_t x) { return (x + 255) & ~size_t(255); };
  const size_t max_inst = (size_t)max_stage_layers * (m.style == ETC_GPT ? 12 : 6) + 6;
  const size_t o_start = 0, o_first = al((size_t)(n_dev + 1) * 4), o_mask = o_first + al((size_t)n_dev * nG * 4),
               o_kstart = o_mask + al((size_t)n_dev * mask_words * 4),
               o_pieces = o_kstart + al((size_t)n_dev * (ETC_NUM_KINDS + 1) * 4);
  const size_t max_total = o_pieces + (size_t)n_dev * n_kinds * max_inst * 5 * sizeof(Piece);   // <= 5 rectangles / instance

  // The lock covers the slab hand-out and, further down, the upload; the build in between runs unlocked, so two host
  // threads can build two layouts side by side (etc_migrate_state does).
  DeviceGuard guard;                                       // the caller's current device is restored on return
  cudaError_t e = guard.err;
  Slab* slab = nullptr;
  if (e == cudaSuccess) { std::lock_guard<std::mutex> lock(g_up_mu); e = slab_acquire(max_total, &slab); }
  if (e != cudaSuccess) { set_error_detail("etc_layout_create staging", e); return ETC_ERR_CUDA; }
  char* host = static_cast<char*>(slab->p);
  int32_t* dev_start = reinterpret_cast<int32_t*>(host + o_start);
  int32_t* first = reinterpret_cast<int32_t*>(host + o_first);
  uint32_t* ltmask = reinterpret_cast<uint32_t*>(host + o_mask);
  int32_t* kind_start = reinterpret_cast<int32_t*>(host + o_kstart);
  Piece* pieces = reinterpret_cast<Piece*>(host + o_pieces);
  memset(first, 0xFF, (size_t)n_dev * nG * 4);
  memset(ltmask, 0, (size_t)n_dev * mask_words * 4);
  int64_t* bufbytes = new int64_t[(size_t)n_dev * ETC_NUM_KINDS]();
  size_t np = 0;
  int32_t n_emb_pieces = 0;
  std::vector<int32_t> grp_pieces((size_t)nG, 0);
  int64_t align_or = 0, total_bytes = 0;

  std::vector<std::vector<Sh>> shr(tp);     // shards of (stage, tp-rank r), in GROUP order: tied replica first
  for (int s = 0; s < pp; ++s) {
    const int l_begin = stage_begin(m.n_layers, *cfg, s), l_end = stage_begin(m.n_layers, *cfg, s + 1);
    // the stage's tensor instances in LOCAL order: pre, layers ascending, post, tied replica (reading A11)
    std::vector<std::pair<int32_t, bool>> inst;
    for (int pass = 0; pass < 3; ++pass)
      for (int t = 0; t < nT; ++t) {
        const LTensor& T = lts[t];
        if (T.where != pass) continue;
        if (pass == 0 && s != 0) continue;
        if (pass == 1 && (T.layer < l_begin || T.layer >= l_end)) continue;
        if (pass == 2 && s != pp - 1) continue;
        inst.push_back({t, false});
      }
    const bool has_replica = two_inst && s == pp - 1;
    if (has_replica) inst.push_back({0, true});
    for (int r = 0; r < tp; ++r) {           // shard geometry depends on (s, r) only
      std::vector<Sh>& sh = shr[r];
      sh.resize(inst.size());
      int64_t pos = 0;
      for (size_t i = 0; i < inst.size(); ++i) {
        const LTensor& T = lts[inst[i].first];
        // start offsets follow LOCAL order; the slot order is GROUP order (the replica, tensor 0, goes first)
        Sh& q = sh[inst[i].second ? 0 : i + (has_replica ? 1 : 0)];
        q.nblk = 1; q.c0 = 0; q.W = T.cols; q.lt = inst[i].first;
        for (int b = 0; b < 3; ++b) { q.rb[b] = q.nr[b] = 0; q.rep[b] = 1; q.rbase[b] = (int16_t)r; }
        q.nr[0] = T.rows;
        switch (T.split) {
          case REPL: q.rep[0] = (int16_t)tp; q.rbase[0] = 0; break;
          case COL: q.nr[0] = T.rows / tp; q.rb[0] = r * q.nr[0]; break;
          case ROW: q.W = T.cols / tp; q.c0 = r * q.W; break;
          case COL2: { const int64_t F = T.rows / 2; q.nblk = 2; q.nr[0] = q.nr[1] = F / tp; q.rb[0] = r * q.nr[0]; q.rb[1] = F + r * q.nr[0]; break; }
          case QKV: qkv_blocks(m, tp, r, q); break;
          default: break;
        }
        int64_t rows = 0;
        for (int b = 0; b < q.nblk; ++b) { q.ls[b] = rows; rows += q.nr[b]; }
        q.n = rows * q.W; q.start = pos; pos += q.n;
        q.flags = (inst[i].second ? PF_POST_COPY : 0) | ((two_inst && inst[i].first == 0) ? 0 : PF_SOLE_INST);
      }
    }
    // The pieces of an UNSHARDED buffer (every kind without the distributed optimizer; PARAM with it) depend on (s, r)
    // only, up to the device id, the kind's group offset and the element size: they are built once per (s, r) and
    // copied with those fields patched for the other DP ranks and kinds (4 ns instead of 15 ns per piece).
    struct Tmpl { size_t begin = 0, count = 0; int64_t es = 0; int kind = -1; int32_t emb = 0; };
    std::vector<Tmpl> tmpl((size_t)tp);
    for (int d = 0; d < dp; ++d)
      for (int r = 0; r < tp; ++r) {
        const int dev = r + tp * (d + dp * s);
        const std::vector<Sh>& sh = shr[r];
        int64_t Lloc = 0; for (const Sh& q : sh) Lloc += q.n;
        dev_start[dev] = (int32_t)np;
        if (d == 0) { for (const Sh& q : sh) ltmask[(size_t)dev * mask_words + q.lt / 32] |= 1u << (q.lt % 32); }
        else memcpy(&ltmask[(size_t)dev * mask_words], &ltmask[(size_t)(r + tp * (dp * s)) * mask_words], (size_t)mask_words * 4);
        for (int kind = 0; kind < ETC_NUM_KINDS; ++kind) {
          kind_start[(size_t)dev * (ETC_NUM_KINDS + 1) + kind] = (int32_t)np;
          if (!((m.kinds >> kind) & 1)) continue;
          const int64_t es = kind == 0 ? m.param_dtype : 4;
          const bool dp_sharded = cfg->dist_opt && dp > 1 && kind >= 1;
          int64_t lo = 0, hi = Lloc;
          Tmpl& tm = tmpl[(size_t)r];
          if (!dp_sharded && tm.kind >= 0) {                 // copy the template of (s, r), patching what differs
            bufbytes[(size_t)dev * ETC_NUM_KINDS + kind] = Lloc * es;
            total_bytes += Lloc * es;
            const int32_t dgrp = (kind - tm.kind) * nT;
            int32_t prev_grp = -1;
            for (size_t i = 0; i < tm.count; ++i) {
              Piece& p = pieces[np];
              p = pieces[tm.begin + i];
              p.dev = dev; p.grp += dgrp; p.d = (int16_t)d; p.boff = p.boff / tm.es * es;
              if (p.grp != prev_grp) { first[(size_t)dev * nG + p.grp] = (int32_t)np; prev_grp = p.grp; }
              grp_pieces[(size_t)p.grp] += 1;
              if (p.W > 1) align_or |= p.boff | ((int64_t)p.W * es) | ((int64_t)p.c0 * es) | ((int64_t)p.nc * es) | (p.f1 * es);
              ++np;
            }
            n_emb_pieces += tm.emb;
            continue;
          }
          const size_t tm_begin = np; const int32_t tm_emb0 = n_emb_pieces;
          if (dp_sharded) {                                  // readings A14 / A28: contiguous flat range of `chunk` elements
            const int64_t unit = (int64_t)dp * std::max(1, cfg->dist_opt_align);
            const int64_t chunk = (Lloc + unit - 1) / unit * std::max(1, cfg->dist_opt_align);
            lo = std::min<int64_t>(Lloc, (int64_t)d * chunk); hi = std::min<int64_t>(Lloc, (int64_t)(d + 1) * chunk);
          }
          bufbytes[(size_t)dev * ETC_NUM_KINDS + kind] = (hi - lo) * es;
          total_bytes += (hi - lo) * es;
          for (const Sh& q : sh) {
            const int64_t a = std::max(lo, q.start) - q.start, b = std::min(hi, q.start + q.n) - q.start;
            if (b <= a) continue;
            const uint16_t flags = q.flags | (dp_sharded ? PF_DP_SHARDED : 0);
            const int32_t grp = kind * nT + q.lt;
            first[(size_t)dev * nG + grp] = (int32_t)np;
            const size_t np_before = np;
            // decompose the held flat range [a,b) of the shard into rectangles of local rows x local cols
            // (head partial row, whole rows cut at the block boundaries, tail partial row: <= 5)
            int64_t rect[5][4]; int nr = 0;
            auto add = [&](int64_t i0, int64_t i1, int64_t j0, int64_t j1) { rect[nr][0] = i0; rect[nr][1] = i1; rect[nr][2] = j0; rect[nr][3] = j1; ++nr; };
            auto add_rows = [&](int64_t i0, int64_t i1) {    // whole local rows [i0,i1), one rectangle per row block
              for (int blk = 0; blk < q.nblk; ++blk) {
                const int64_t x0 = std::max(i0, q.ls[blk]), x1 = std::min(i1, q.ls[blk] + q.nr[blk]);
                if (x1 > x0) add(x0, x1, 0, q.W);
              }
            };
            if (a == 0 && b == q.n) add_rows(0, q.n / q.W);  // whole shard (the common case)
            else {
              const int64_t ia = a / q.W, ja = a % q.W, ib = b / q.W, jb = b % q.W;
              if (ia == ib) add(ia, ia + 1, ja, jb);
              else {
                int64_t body0 = ia;
                if (ja > 0) { add(ia, ia + 1, ja, q.W); body0 = ia + 1; }
                if (ib > body0) add_rows(body0, ib);
                if (jb > 0) add(ib, ib + 1, 0, jb);
              }
            }
            for (int k = 0; k < nr; ++k) {
              const int64_t i0 = rect[k][0], i1 = rect[k][1], j0 = rect[k][2], j1 = rect[k][3];
              int blk = 0;
              while (blk + 1 < q.nblk && i0 >= q.ls[blk] + q.nr[blk]) ++blk;
              Piece& p = pieces[np++];
              p.dev = dev; p.grp = grp;
              p.r0 = (int32_t)(q.rb[blk] + (i0 - q.ls[blk])); p.nr = (int32_t)(i1 - i0);
              p.c0 = (int32_t)(q.c0 + j0); p.nc = (int32_t)(j1 - j0);
              p.lrow0 = (int32_t)i0; p.lcol0 = (int32_t)j0; p.W = (int32_t)q.W;
              p.s = (int16_t)s; p.r = (int16_t)r; p.d = (int16_t)d; p.flags = flags;
              p.rep = q.rep[blk]; p.rbase = q.rbase[blk];
              p.boff = (q.start + i0 * q.W + j0 - lo) * es;
              p.f0 = a; p.f1 = b;
              // a one-column tensor (a bias stored n x 1) cannot be cut by columns: its slices are contiguous runs whatever
              // their alignment, so it does not count (see etc_layout::aligned16)
              if (p.W > 1) align_or |= p.boff | ((int64_t)p.W * es) | ((int64_t)p.c0 * es) | ((int64_t)p.nc * es) | (a * es) | (b * es);
            }
            grp_pieces[(size_t)grp] += (int32_t)(np - np_before);
            if (q.lt == 0 || (!m.tied_embeddings && q.lt == nT - 1)) n_emb_pieces += (int32_t)(np - np_before);
          }
          if (!dp_sharded) { tm.begin = tm_begin; tm.count = np - tm_begin; tm.es = es; tm.kind = kind; tm.emb = n_emb_pieces - tm_emb0; }
        }
        kind_start[(size_t)dev * (ETC_NUM_KINDS + 1) + ETC_NUM_KINDS] = (int32_t)np;
      }
  }
  dev_start[n_dev] = (int32_t)np;
  int32_t max_dev_pieces = 0;
  for (int i = 0; i < n_dev; ++i) max_dev_pieces = std::max(max_dev_pieces, dev_start[i + 1] - dev_start[i]);
  const size_t total = o_pieces + al(np * sizeof(Piece));

  etc_layout* L = new etc_layout();
  L->model = m; L->cfg = *cfg; L->h_buffer_bytes = bufbytes; L->max_dev_pieces = max_dev_pieces;
  L->vocab_rows = (int32_t)vocab_rows(m, *cfg); L->lm_head_id = m.tied_embeddings ? -1 : nT - 1; L->n_emb_pieces = n_emb_pieces;
  L->grp_pieces = std::move(grp_pieces); L->aligned16 = (align_or & 15) == 0; L->total_bytes = total_bytes;
  for (int s = 0; s <= pp; ++s) L->stage_first.push_back(stage_begin(m.n_layers, *cfg, s));
  std::lock_guard<std::mutex> lock(g_up_mu);               // the upload stream and the slab's state
  e = cudaMallocAsync(&L->d_blob, total, g_up_stream);
  // a DMA copy on the private upload stream: it runs beside the copy kernels of a migration in flight (a copy kernel
  // here was measured to wait for them: 0.16 -> 1.7 ms per layout pair on c2).  No host wait: readers wait for `ready`.
  if (e == cudaSuccess) e = cudaMemcpyAsync(L->d_blob, host, total, cudaMemcpyHostToDevice, g_up_stream);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&L->ready, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventRecord(L->ready, g_up_stream);
  if (e == cudaSuccess) { e = cudaEventRecord(slab->done, g_up_stream); slab->in_flight = e == cudaSuccess; }
  slab->busy = false;
  if (e != cudaSuccess) {
    set_error_detail("etc_layout_create upload", e);
    cudaStreamSynchronize(g_up_stream);                    // the slab may still be being read
    if (L->d_blob) cudaFreeAsync(L->d_blob, g_up_stream);
    if (L->ready) cudaEventDestroy(L->ready);
    delete[] bufbytes; delete L;
    return ETC_ERR_CUDA;
  }
  char* base = (char*)L->d_blob;
  L->t.pieces = (const Piece*)(base + o_pieces);
  L->t.dev_start = (const int32_t*)(base + o_start);
  L->t.first = (const int32_t*)(base + o_first);
  L->t.ltmask = (const uint32_t*)(base + o_mask);
  L->t.kind_start = (const int32_t*)(base + o_kstart);
  L->t.n_dev = n_dev; L->t.n_grp = nG; L->t.n_tensors = nT; L->t.mask_words = mask_words;
  L->t.n_pieces = (int32_t)np;
  L->t.tp = tp; L->t.pp = pp; L->t.dp = dp;
  for (int k = 0; k < ETC_NUM_KINDS; ++k) L->t.elem_bytes[k] = k == 0 ? m.param_dtype : 4;
  *out = L;
  return ETC_OK;
}

extern "C" void etc_layout_destroy(etc_layout* L) {
  if (!L) return;
  DeviceGuard device_guard;
  // stream-ordered free, ordered after every kernel already enqueued on any stream that read the tables
  if (L->d_blob) cudaFreeAsync(L->d_blob, L->streams.join(g_up_stream));
  if (L->ready) cudaEventDestroy(L->ready);
  delete[] L->h_buffer_bytes;
  delete L;
}

extern "C" int32_t etc_layout_num_devices(const etc_layout* L) { return L ? L->t.n_dev : ETC_ERR_INVALID_ARG; }
extern "C" int64_t etc_layout_num_pieces(const etc_layout* L) { return L ? L->t.n_pieces : ETC_ERR_INVALID_ARG; }
extern "C" int64_t etc_layout_buffer_bytes(const etc_layout* L, int32_t dev, int32_t kind) {
  if (!L || dev < 0 || dev >= L->t.n_dev || kind < 0 || kind >= ETC_NUM_KINDS) return ETC_ERR_INVALID_ARG;
  return L->h_buffer_bytes[(size_t)dev * ETC_NUM_KINDS + kind];
}

extern "C" const char* etc_status_string(etc_status s) {
  switch (s) {
    case ETC_OK: return "ETC_OK";
    case ETC_ERR_INVALID_ARG: return "ETC_ERR_INVALID_ARG";
    case ETC_ERR_INDIVISIBLE: return "ETC_ERR_INDIVISIBLE";
    case ETC_ERR_MISMATCH: return "ETC_ERR_MISMATCH";
    case ETC_ERR_BAD_MAP: return "ETC_ERR_BAD_MAP";
    case ETC_ERR_WORKSPACE: return "ETC_ERR_WORKSPACE";
    case ETC_ERR_UNSUPPORTED: return "ETC_ERR_UNSUPPORTED";
    case ETC_ERR_CUDA: return "ETC_ERR_CUDA";
    case ETC_ERR_UNRECOVERABLE: return "ETC_ERR_UNRECOVERABLE";
    default: return "ETC_ERR_UNKNOWN";
  }
}
extern "C" const char* etc_last_error_detail(void) { return g_detail.c_str(); }
extern "C" int64_t etc_kernel_launches(void) { return __atomic_load_n(&g_launches, __ATOMIC_RELAXED); }
