// layout.cu — (a1) layout descriptor: (model_desc, parallel_cfg) -> index rectangles ("pieces") of every state tensor
// on every device, uploaded once.  Host-side integer bookkeeping only (PAPER.md:106 workload abstraction; :110 "each
// device can derive its workload following these rules"; :199 TP slices -> explicit split types, reading A8).
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <ctime>
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
void clear_error_detail() { g_detail.clear(); }
void count_launch(int n) { __atomic_add_fetch(&g_launches, (long long)n, __ATOMIC_RELAXED); }
int current_device() { return g_device; }

struct LTensor { int64_t rows, cols; int32_t split, where, layer; };   // where: 0 pre, 1 layer, 2 post

// Logical tensor list in id order.  QKV rows are in KV-group order, so an equal row split
// is the GQA-aware split as long as n_kv_heads % tp == 0 (reading A10); SwiGLU fc1 = [gate; up] is COL2.
static std::vector<LTensor> logical_tensors(const etc_model_desc& m) {
  std::vector<LTensor> v;
  const int64_t h = m.hidden, d = m.head_dim, f = m.ffn_hidden;
  const int64_t qkv = (int64_t(m.n_q_heads) + 2 * int64_t(m.n_kv_heads)) * d, qd = int64_t(m.n_q_heads) * d;
  v.push_back({m.vocab, h, COL, 0, -1});
  if (m.style == ETC_GPT && m.max_pos > 0) v.push_back({m.max_pos, h, REPL, 0, -1});
  for (int l = 0; l < m.n_layers; ++l) {
    if (m.style == ETC_GPT) {
      v.push_back({1, h, REPL, 1, l}); v.push_back({1, h, REPL, 1, l});          // ln1 w,b
      v.push_back({qkv, h, COL, 1, l}); v.push_back({qkv, 1, COL, 1, l});        // qkv w,b
      v.push_back({h, qd, ROW, 1, l}); v.push_back({1, h, REPL, 1, l});          // proj w,b
      v.push_back({1, h, REPL, 1, l}); v.push_back({1, h, REPL, 1, l});          // ln2 w,b
      v.push_back({f, h, COL, 1, l}); v.push_back({f, 1, COL, 1, l});            // fc1 w,b
      v.push_back({h, f, ROW, 1, l}); v.push_back({1, h, REPL, 1, l});           // fc2 w,b
    } else {
      v.push_back({1, h, REPL, 1, l});                                           // ln1 w
      v.push_back({qkv, h, COL, 1, l});                                          // qkv w
      v.push_back({h, qd, ROW, 1, l});                                           // proj w
      v.push_back({1, h, REPL, 1, l});                                           // ln2 w
      v.push_back({2 * f, h, COL2, 1, l});                                       // fc1 w = [gate; up]
      v.push_back({h, f, ROW, 1, l});                                            // fc2 w
    }
  }
  v.push_back({1, h, REPL, 2, -1});                                              // final_ln w
  if (m.style == ETC_GPT) v.push_back({1, h, REPL, 2, -1});                      // final_ln b
  if (!m.tied_embeddings) v.push_back({m.vocab, h, COL, 2, -1});                 // lm_head
  return v;
}

static etc_status validate(const etc_model_desc* m, const etc_parallel_cfg* c) {
  if (!m || !c) return ETC_ERR_INVALID_ARG;
  if (c->tp < 1 || c->pp < 1 || c->dp < 1 || (c->dist_opt != 0 && c->dist_opt != 1)) return ETC_ERR_INVALID_ARG;
  if (m->style != ETC_GPT && m->style != ETC_LLAMA) return ETC_ERR_INVALID_ARG;
  if (m->n_layers < 1 || m->hidden < 1 || m->n_q_heads < 1 || m->n_kv_heads < 1 || m->head_dim < 1 ||
      m->ffn_hidden < 1 || m->vocab < 1 || m->max_pos < 0) return ETC_ERR_INVALID_ARG;
  if (m->param_dtype != ETC_BF16 && m->param_dtype != ETC_FP32) return ETC_ERR_INVALID_ARG;
  if (m->kinds <= 0 || m->kinds > 15) return ETC_ERR_INVALID_ARG;
  if (m->tied_embeddings != 0 && m->tied_embeddings != 1) return ETC_ERR_INVALID_ARG;
  if (m->n_q_heads % m->n_kv_heads) return ETC_ERR_INVALID_ARG;
  if (int64_t(c->tp) * c->pp * c->dp > 32767) return ETC_ERR_INVALID_ARG;
  if (c->tp > m->n_kv_heads) return ETC_ERR_UNSUPPORTED;
  if (m->n_layers % c->pp || m->n_kv_heads % c->tp || m->ffn_hidden % c->tp || m->vocab % c->tp)
    return ETC_ERR_INDIVISIBLE;
  return ETC_OK;
}

struct Inst { int32_t lt; bool post_copy; };

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

extern "C" etc_status etc_layout_create(const etc_model_desc* model, const etc_parallel_cfg* cfg, etc_layout** out) {
  clear_error_detail();
  if (!out) return ETC_ERR_INVALID_ARG;
  etc_status st = validate(model, cfg);
  if (st != ETC_OK) return st;
  if (getenv("ETC_TIME_LAYOUT")) { timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts); fprintf(stderr, "layout start at %ld.%09ld\n", ts.tv_sec, ts.tv_nsec); }
  const etc_model_desc& m = *model;
  const int tp = cfg->tp, pp = cfg->pp, dp = cfg->dp;
  const int n_dev = tp * pp * dp;
  const std::vector<LTensor> lts = logical_tensors(m);
  const int nT = (int)lts.size(), nG = nT * ETC_NUM_KINDS;
  const int per_stage = m.n_layers / pp;
  const bool two_inst = m.tied_embeddings && pp > 1;     // word_embeddings held by first AND last stage

  std::vector<Piece> pieces;
  std::vector<int64_t> bufbytes((size_t)n_dev * ETC_NUM_KINDS, 0);
  std::vector<int32_t> dev_start(n_dev + 1, 0);
  const int mask_words = (nT + 31) / 32;
  std::vector<uint32_t> ltmask((size_t)n_dev * mask_words, 0u);

  for (int dev = 0; dev < n_dev; ++dev) {
    const int r = dev % tp, d = (dev / tp) % dp, s = dev / (tp * dp);
    dev_start[dev] = (int32_t)pieces.size();
    // the stage's tensor instances in local order: pre, layers ascending, post, tied replica
    std::vector<Inst> inst;
    for (int pass = 0; pass < 3; ++pass)
      for (int t = 0; t < nT; ++t) {
        const LTensor& T = lts[t];
        if (T.where != pass) continue;
        if (pass == 0 && s != 0) continue;
        if (pass == 1 && (T.layer < s * per_stage || T.layer >= (s + 1) * per_stage)) continue;
        if (pass == 2 && s != pp - 1) continue;
        inst.push_back({t, false});
      }
    if (two_inst && s == pp - 1) inst.push_back({0, true});
    // shard geometry + start offsets in the (s,r) local flat space
    struct Sh { int64_t start, n, rb[2], nrb, c0, W; int nblk; };
    std::vector<Sh> sh(inst.size());
    int64_t Lloc = 0;
    for (size_t i = 0; i < inst.size(); ++i) {
      const LTensor& T = lts[inst[i].lt];
      Sh& q = sh[i];
      q.nblk = 1; q.rb[0] = q.rb[1] = 0; q.nrb = T.rows; q.c0 = 0; q.W = T.cols;
      switch (T.split) {
        case COL: q.nrb = T.rows / tp; q.rb[0] = r * q.nrb; break;
        case ROW: q.W = T.cols / tp; q.c0 = r * q.W; break;
        case COL2: { const int64_t F = T.rows / 2; q.nblk = 2; q.nrb = F / tp; q.rb[0] = r * q.nrb; q.rb[1] = F + r * q.nrb; break; }
        default: break;
      }
      q.n = (int64_t)q.nblk * q.nrb * q.W; q.start = Lloc; Lloc += q.n;
    }
    const size_t dev_first_piece = pieces.size();
    for (int kind = 0; kind < ETC_NUM_KINDS; ++kind) {
      if (!((m.kinds >> kind) & 1)) continue;
      const int64_t es = kind == 0 ? m.param_dtype : 4;
      const bool dp_sharded = cfg->dist_opt && dp > 1 && kind >= 1;
      int64_t lo = 0, hi = Lloc;
      if (dp_sharded) {                                      // reading A14: contiguous flat range, chunk = ceil(Lloc/dp)
        const int64_t chunk = (Lloc + dp - 1) / dp;
        lo = std::min<int64_t>(Lloc, (int64_t)d * chunk); hi = std::min<int64_t>(Lloc, (int64_t)(d + 1) * chunk);
      }
      bufbytes[(size_t)dev * ETC_NUM_KINDS + kind] = (hi - lo) * es;
      for (size_t i = 0; i < inst.size(); ++i) {
        const Sh& q = sh[i];
        const LTensor& T = lts[inst[i].lt];
        const int64_t a = std::max(lo, q.start) - q.start, b = std::min(hi, q.start + q.n) - q.start;
        if (b <= a) continue;
        uint16_t flags = 0;
        if (inst[i].post_copy) flags |= PF_POST_COPY;
        if (!(two_inst && inst[i].lt == 0)) flags |= PF_SOLE_INST;
        if (T.split != REPL) flags |= PF_TP_SHARDED;
        if (dp_sharded) flags |= PF_DP_SHARDED;
        // decompose the held flat range [a,b) of the shard into rectangles of local rows x local cols
        struct LR { int64_t i0, i1, j0, j1; };
        LR rects[4]; int nr = 0;
        const int64_t ia = a / q.W, ja = a % q.W, ib = b / q.W, jb = b % q.W;
        if (ia == ib) rects[nr++] = {ia, ia + 1, ja, jb};
        else {
          int64_t body0 = ia;
          if (ja > 0) { rects[nr++] = {ia, ia + 1, ja, q.W}; body0 = ia + 1; }
          if (ib > body0) {
            if (q.nblk == 2 && body0 < q.nrb && ib > q.nrb) {          // body spans the gate/up block boundary
              rects[nr++] = {body0, q.nrb, 0, q.W}; rects[nr++] = {q.nrb, ib, 0, q.W};
            } else rects[nr++] = {body0, ib, 0, q.W};
          }
          if (jb > 0) rects[nr++] = {ib, ib + 1, 0, jb};
        }
        for (int k = 0; k < nr; ++k) {
          const LR& R = rects[k];
          const int blk = (int)(R.i0 / q.nrb);
          Piece p;
          p.dev = dev; p.grp = kind * nT + inst[i].lt;
          p.r0 = (int32_t)(q.rb[blk] + R.i0 % q.nrb); p.nr = (int32_t)(R.i1 - R.i0);
          p.c0 = (int32_t)(q.c0 + R.j0); p.nc = (int32_t)(R.j1 - R.j0);
          p.lrow0 = (int32_t)R.i0; p.lcol0 = (int32_t)R.j0; p.W = (int32_t)q.W;
          p.s = (int16_t)s; p.r = (int16_t)r; p.d = (int16_t)d; p.flags = flags;
          p.boff = (q.start + R.i0 * q.W + R.j0 - lo) * es;
          p.f0 = a; p.f1 = b;
          pieces.push_back(p);
        }
        ltmask[(size_t)dev * mask_words + inst[i].lt / 32] |= 1u << (inst[i].lt % 32);
      }
    }
    std::stable_sort(pieces.begin() + dev_first_piece, pieces.end(),
                     [](const Piece& x, const Piece& y) { return x.grp < y.grp; });
  }
  dev_start[n_dev] = (int32_t)pieces.size();
  if (pieces.size() > (size_t)INT32_MAX) return ETC_ERR_INVALID_ARG;

  std::vector<int32_t> first((size_t)n_dev * nG, -1);
  for (int32_t i = (int32_t)pieces.size() - 1; i >= 0; --i) first[(size_t)pieces[i].dev * nG + pieces[i].grp] = i;

  // one device blob: pieces | dev_start | first | ltmask
  auto al = [](size_t x) { return (x + 255) & ~size_t(255); };
  const size_t o_pieces = 0, o_start = al(pieces.size() * sizeof(Piece)),
               o_first = o_start + al(dev_start.size() * 4), o_mask = o_first + al(first.size() * 4),
               total = o_mask + al(ltmask.size() * 4);
  std::vector<char> host(total, 0);
  if (!pieces.empty()) memcpy(host.data() + o_pieces, pieces.data(), pieces.size() * sizeof(Piece));
  memcpy(host.data() + o_start, dev_start.data(), dev_start.size() * 4);
  memcpy(host.data() + o_first, first.data(), first.size() * 4);
  memcpy(host.data() + o_mask, ltmask.data(), ltmask.size() * 4);

  if (getenv("ETC_TIME_LAYOUT")) { timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts); fprintf(stderr, "layout host build done at %ld.%09ld pieces=%zu total=%zu\n", ts.tv_sec, ts.tv_nsec, pieces.size(), total); }
  etc_layout* L = new etc_layout();
  L->model = m; L->cfg = *cfg;
  cudaError_t e = cudaSetDevice(current_device());
  if (e == cudaSuccess) e = cudaMalloc(&L->d_blob, total);
  if (e == cudaSuccess) e = cudaMemcpy(L->d_blob, host.data(), total, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    set_error_detail("etc_layout_create upload", e);
    if (L->d_blob) cudaFree(L->d_blob);
    delete L;
    return ETC_ERR_CUDA;
  }
  char* base = (char*)L->d_blob;
  L->t.pieces = (const Piece*)(base + o_pieces);
  L->t.dev_start = (const int32_t*)(base + o_start);
  L->t.first = (const int32_t*)(base + o_first);
  L->t.ltmask = (const uint32_t*)(base + o_mask);
  L->t.n_dev = n_dev; L->t.n_grp = nG; L->t.n_tensors = nT; L->t.mask_words = mask_words;
  L->t.n_pieces = (int32_t)pieces.size();
  L->t.tp = tp; L->t.pp = pp; L->t.dp = dp;
  for (int k = 0; k < ETC_NUM_KINDS; ++k) L->t.elem_bytes[k] = k == 0 ? m.param_dtype : 4;
  L->h_buffer_bytes = new int64_t[bufbytes.size()];
  memcpy(L->h_buffer_bytes, bufbytes.data(), bufbytes.size() * sizeof(int64_t));
  *out = L;
  return ETC_OK;
}

extern "C" void etc_layout_destroy(etc_layout* L) {
  if (!L) return;
  if (L->d_blob) cudaFree(L->d_blob);
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
    default: return "ETC_ERR_UNKNOWN";
  }
}
extern "C" const char* etc_last_error_detail(void) { return g_detail.c_str(); }
extern "C" int64_t etc_kernel_launches(void) { return __atomic_load_n(&g_launches, __ATOMIC_RELAXED); }
