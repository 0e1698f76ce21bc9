/*
 * etc_oracle.c — TEST INFRASTRUCTURE ONLY.  Plain, slow, element-by-element CPU definition of the hot path of
 * ETC's checkpoint-free migration (arxiv/paper_2607_04749; citations are PAPER.md line numbers).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this.
 * It shares no code, header, table or helper with paper_2607_04749_b200/ (the CUDA path) and never calls it.
 *
 * What it defines:
 *   - the logical model (tensor list + TP split type, reading A8/A10) and the Megatron-style DPxTPxPP layout:
 *     global_of(dev, kind, local) -> (tensor, row, col)   and   holders_of(kind, tensor, row, col) -> {(dev, local)}
 *   - hold[o], need[n], overlap[n][o]  (paper's cost c[n][o] = need[n] - overlap[n][o])
 *   - the sketch objective, by brute force over every injective device map and by a plain O(k^3) Hungarian on the
 *     zero-padded square matrix (Algorithm 1)
 *   - the source of every needed element (reading A6), the traffic matrix T, and the element-wise migration
 *     (Send/Recv/Refer semantics of PAPER.md:193-201: every destination element is fetched from its one source).
 *
 * Everything is integer / raw bytes: parity with the CUDA path is bit-exact ("bit-exact fidelity").
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): P1 paper's worked example PAPER.md:108, P2 identity
 * reconfiguration, P3 sum identities, P4 reassembly, P5 brute force vs Hungarian, P6 SciPy linear_sum_assignment,
 * P7 PP/TP merge rule, P8/P9 stamped payloads, P10 exactly-once, P11 closed forms, P12 swept tiny layouts, and
 * holders_of checked against brute-force inversion of global_of.  Parity with the paper itself is "unpinned" for
 * the choices the paper leaves open (A9-A14: rank order, QKV/SwiGLU local order, tied embeddings, dist-opt ranges);
 * those are pinned only against DESIGN.md's stated readings.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_KINDS 4
enum { ORC_REPL = 0, ORC_COL = 1, ORC_ROW = 2, ORC_COL2 = 3, ORC_QKV = 4 };
enum { ORC_PRE = 0, ORC_LAYER = 1, ORC_POST = 2 };
enum { ORC_OK = 0, ORC_ERR_ARG = -1, ORC_ERR_INDIVISIBLE = -2, ORC_ERR_UNSUPPORTED = -6, ORC_ERR_UNRECOVERABLE = -8 };

typedef struct {
  int32_t style;       /* 0 = GPT (LayerNorm+bias, linear bias, learned pos-emb); 1 = LLaMA (RMSNorm, SwiGLU) */
  int32_t n_layers, hidden, n_q_heads, n_kv_heads, head_dim, ffn_hidden, vocab, max_pos;
  int32_t tied;        /* 1: output layer shares word_embeddings (replica on the last PP stage when pp > 1) */
  int32_t param_bytes; /* element size of kind PARAM: 2 (bf16) or 4 (fp32) */
  int32_t kinds;       /* bitmask over kinds 0..3 = PARAM, MASTER, ADAM_M, ADAM_V */
  int32_t qkv_order;   /* logical row order of the fused QKV tensor (readings A10, A29): 0 = KV-group order (per group:
                          its q heads, K, V); 1 = [Q; K; V] (all q heads, then all k heads, then all v heads) */
} orc_model;

/* pp_first / pp_last: layers on the first / last pipeline stage (0 = not set), reading A27 (uneven pipeline split) */
/* dist_opt_align (reading A28, f3): the DP shard size of the distributed optimizer is rounded up to a multiple of this
 * many elements (0 or 1 = no rounding), as Megatron-LM pads its buffers so that every DP shard is aligned */
/* vocab_divisor (reading A31, f3): > 0 pads the vocabulary dimension of word_embeddings / lm_head to a multiple of
 * vocab_divisor * tp rows (Megatron-LM's --make-vocab-size-divisible-by); the padding rows are stored like any other
 * row.  0 = no padding: vocab % tp == 0 is required (reading A12) */
typedef struct { int32_t tp, pp, dp, dist_opt, pp_first, pp_last, dist_opt_align, vocab_divisor; } orc_cfg;

typedef struct { int64_t rows, cols; int32_t split, where, layer; } orc_lt;   /* one logical tensor */

/* one tensor shard inside the local flat space of a (stage, tp-rank) pair */
typedef struct {
  int32_t lt;          /* logical tensor id */
  int32_t post_copy;   /* 1: this is the tied replica of word_embeddings held by the last stage */
  int64_t start, n;    /* position and element count inside the local flat space */
  int32_t nblk;        /* row blocks, stored one after the other (COL2: gate, up; QKV: up to 3, readings A29/A30) */
  int64_t rb[3], nr[3]; /* first logical row and number of rows of each block */
  int32_t rep[3];      /* how many TP ranks hold each element of the block (1 = TP-sharded, tp = replicated) */
  int64_t c0, W;       /* first logical column, local row length */
} orc_shard;

typedef struct {
  orc_model m; orc_cfg c;
  int32_t n_lt; orc_lt* lt;
  int32_t* n_sh; orc_shard** sh; int64_t* Lloc;      /* indexed by s*tp + r */
  int32_t* idx;        /* [pp][n_lt]: position of tensor lt in stage s's shard list (same for every r), or -1 */
  int32_t* tied_idx;   /* [pp]: position of the tied word_embeddings replica in stage s's list, or -1 */
  uint8_t* failed;     /* optional [n_dev]: 1 = the device failed and its state is lost (reading A26), NULL = none */
} orc_layout;

/* ---------------------------------------------------------------- logical model */
/* rows of the embedding tensors in a layout: the padded vocabulary (reading A31) */
static int64_t orc_vocab_rows(const orc_model* m, const orc_cfg* c) {
  if (!c || c->vocab_divisor <= 0) return m->vocab;
  int64_t unit = (int64_t)c->vocab_divisor * c->tp;
  return ((int64_t)m->vocab + unit - 1) / unit * unit;
}

/* c == NULL: the unpadded logical model */
static int orc_logical(const orc_model* m, const orc_cfg* c, orc_lt* out) {
  int n = 0;
  const int64_t V = orc_vocab_rows(m, c);
  const int64_t h = m->hidden, d = m->head_dim;
  const int64_t qkv = ((int64_t)m->n_q_heads + 2 * (int64_t)m->n_kv_heads) * d;
  const int64_t qd = (int64_t)m->n_q_heads * d, f = m->ffn_hidden;
#define ADD(R, C, S, WH, LY) do { if (out) { out[n].rows = (R); out[n].cols = (C); out[n].split = (S); \
                                  out[n].where = (WH); out[n].layer = (LY); } n++; } while (0)
  ADD(V, h, ORC_COL, ORC_PRE, -1);                               /* word_embeddings */
  if (m->style == 0 && m->max_pos > 0) ADD(m->max_pos, h, ORC_REPL, ORC_PRE, -1);   /* position_embeddings */
  for (int l = 0; l < m->n_layers; l++) {
    if (m->style == 0) {
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* ln1.weight */
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* ln1.bias */
      ADD(qkv, h, ORC_QKV, ORC_LAYER, l);     /* qkv.weight (A10, A29, A30) */
      ADD(qkv, 1, ORC_QKV, ORC_LAYER, l);     /* qkv.bias */
      ADD(h, qd, ORC_ROW, ORC_LAYER, l);      /* proj.weight */
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* proj.bias */
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* ln2.weight */
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* ln2.bias */
      ADD(f, h, ORC_COL, ORC_LAYER, l);       /* fc1.weight */
      ADD(f, 1, ORC_COL, ORC_LAYER, l);       /* fc1.bias */
      ADD(h, f, ORC_ROW, ORC_LAYER, l);       /* fc2.weight */
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* fc2.bias */
    } else {
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* ln1.weight */
      ADD(qkv, h, ORC_QKV, ORC_LAYER, l);     /* qkv.weight */
      ADD(h, qd, ORC_ROW, ORC_LAYER, l);      /* proj.weight */
      ADD(1, h, ORC_REPL, ORC_LAYER, l);      /* ln2.weight */
      ADD(2 * f, h, ORC_COL2, ORC_LAYER, l);  /* fc1.weight = [gate; up] */
      ADD(h, f, ORC_ROW, ORC_LAYER, l);       /* fc2.weight */
    }
  }
  ADD(1, h, ORC_REPL, ORC_POST, -1);                             /* final_ln.weight */
  if (m->style == 0) ADD(1, h, ORC_REPL, ORC_POST, -1);          /* final_ln.bias */
  if (!m->tied) ADD(V, h, ORC_COL, ORC_POST, -1);                /* lm_head */
#undef ADD
  return n;
}

int32_t orc_num_logical(const orc_model* m) { return orc_logical(m, NULL, NULL); }

/* rows[i], cols[i], split[i], where[i], layer[i] for every logical tensor */
int32_t orc_logical_info_cfg(const orc_model* m, const orc_cfg* c, int64_t* rows, int64_t* cols, int32_t* split,
                             int32_t* where, int32_t* layer);
int32_t orc_logical_info(const orc_model* m, int64_t* rows, int64_t* cols, int32_t* split, int32_t* where,
                         int32_t* layer) {
  return orc_logical_info_cfg(m, NULL, rows, cols, split, where, layer);
}
/* the same with the embedding rows of a given parallel configuration (padded vocabulary, reading A31) */
int32_t orc_logical_info_cfg(const orc_model* m, const orc_cfg* c, int64_t* rows, int64_t* cols, int32_t* split,
                             int32_t* where, int32_t* layer) {
  int n = orc_logical(m, c, NULL);
  orc_lt* t = (orc_lt*)malloc(sizeof(orc_lt) * (size_t)n);
  orc_logical(m, c, t);
  for (int i = 0; i < n; i++) {
    rows[i] = t[i].rows; cols[i] = t[i].cols; split[i] = t[i].split; where[i] = t[i].where; layer[i] = t[i].layer;
  }
  free(t);
  return n;
}

static int orc_elem_bytes(const orc_model* m, int kind) { return kind == 0 ? m->param_bytes : 4; }
int32_t orc_kind_bytes(const orc_model* m, int32_t kind) { return orc_elem_bytes(m, kind); }

/* First layer of pipeline stage s (s = pp gives n_layers).  Even split ("divisible by PP sizes") unless
 * pp_first / pp_last fix the layer count of the first / last stage (reading A27, as Megatron-LM's
 * --decoder-first/last-pipeline-num-layers): the remaining layers are split evenly over the remaining stages.
 * Returns -1 if the split is impossible (indivisible, or a stage would be empty), -2 on nonsense arguments. */
static int orc_stage_begin(int n_layers, const orc_cfg* c, int s) {
  int first = c->pp_first, last = c->pp_last, pp = c->pp;
  if (first < 0 || last < 0) return -2;
  if ((first || last) && pp < 2) return -2;
  int mid_stages = pp - (first ? 1 : 0) - (last ? 1 : 0), mid_layers = n_layers - first - last;
  if (mid_stages < 0 || mid_layers < 0) return -1;
  if (mid_stages == 0) { if (mid_layers != 0) return -1; }
  else if (mid_layers % mid_stages || mid_layers / mid_stages < 1) return -1;
  int per = mid_stages ? mid_layers / mid_stages : 0;
  if (s <= 0) return 0;
  if (s >= pp) return n_layers;
  if (first) return first + (s - 1) * per;
  return s * per;
}

/* divisibility rules (layers divisible by PP, hidden by TP; A7, A10, A12) */
static int orc_validate(const orc_model* m, const orc_cfg* c) {
  if (!m || !c) return ORC_ERR_ARG;
  if (c->tp < 1 || c->pp < 1 || c->dp < 1 || c->dist_opt_align < 0 || c->vocab_divisor < 0) return ORC_ERR_ARG;
  if (m->n_layers < 1 || m->hidden < 1 || m->n_q_heads < 1 || m->n_kv_heads < 1 || m->head_dim < 1 ||
      m->ffn_hidden < 1 || m->vocab < 1 || m->max_pos < 0) return ORC_ERR_ARG;
  if (m->param_bytes != 2 && m->param_bytes != 4) return ORC_ERR_ARG;
  if (m->kinds <= 0 || m->kinds > 15) return ORC_ERR_ARG;
  if (m->n_q_heads % m->n_kv_heads) return ORC_ERR_ARG;
  if (m->qkv_order != 0 && m->qkv_order != 1) return ORC_ERR_ARG;
  if (c->tp > m->n_kv_heads) {                                 /* KV-head replication (reading A30) */
    int rep = c->tp / m->n_kv_heads;
    if (c->tp % m->n_kv_heads || (m->n_q_heads / m->n_kv_heads) % rep) return ORC_ERR_UNSUPPORTED;
  }
  if (orc_stage_begin(m->n_layers, c, 0) < 0) return orc_stage_begin(m->n_layers, c, 0) == -2 ? ORC_ERR_ARG : ORC_ERR_INDIVISIBLE;
  if (c->tp <= m->n_kv_heads && m->n_kv_heads % c->tp) return ORC_ERR_INDIVISIBLE;
  if (m->ffn_hidden % c->tp) return ORC_ERR_INDIVISIBLE;
  if (c->vocab_divisor == 0 && m->vocab % c->tp) return ORC_ERR_INDIVISIBLE;   /* A12; with padding (A31) it always divides */
  return ORC_OK;
}

/* ---------------------------------------------------------------- layout */
/* TP shard of logical tensor t on TP rank r: an ordered list of row blocks x a column range.
 * QKV (readings A10, A29, A30): with q = n_q heads, k = n_kv heads, d rows per head, qpg = q/k q heads per KV group.
 *   tp <= k (each rank holds whole groups, kpr = k/tp of them):
 *     order 0 (group order, group g = rows [g*(qpg+2)*d, (g+1)*(qpg+2)*d)): one block, groups [r*kpr, (r+1)*kpr)
 *     order 1 ([Q;K;V]): three blocks: q heads [r*q/tp, (r+1)*q/tp), k heads [r*kpr, (r+1)*kpr), v heads likewise
 *   tp > k (KV-head replication, rep = tp/k ranks share group g = r/rep; rank r holds qpr = qpg/rep q heads of it,
 *           the j-th share with j = r % rep, and the WHOLE K and V head of the group):
 *     order 0: two blocks: q rows [g*(qpg+2)*d + j*qpr*d, +qpr*d), then the K,V rows [g*(qpg+2)*d + qpg*d, +2d)
 *     order 1: three blocks: q heads [r*qpr, (r+1)*qpr), k head g, v head g
 *   K and V blocks of the replicated case are held by rep ranks (rep[] = tp/k), everything else by one. */
static void orc_make_shard(const orc_model* m, const orc_lt* t, int lt, int post_copy, int tp, int r, orc_shard* s) {
  s->lt = lt; s->post_copy = post_copy; s->nblk = 1; s->c0 = 0; s->W = t->cols;
  for (int b = 0; b < 3; b++) { s->rb[b] = 0; s->nr[b] = 0; s->rep[b] = 1; }
  s->nr[0] = t->rows;
  switch (t->split) {
    case ORC_REPL: s->rep[0] = tp; break;                                       /* whole tensor on every rank */
    case ORC_COL:  s->nr[0] = t->rows / tp; s->rb[0] = r * s->nr[0]; break;     /* rows / tp */
    case ORC_ROW:  s->W = t->cols / tp; s->c0 = r * s->W; break;                /* cols / tp */
    case ORC_COL2: { int64_t F = t->rows / 2; s->nblk = 2; s->nr[0] = s->nr[1] = F / tp;   /* gate block, then up block */
                     s->rb[0] = r * s->nr[0]; s->rb[1] = F + r * s->nr[0]; break; }
    case ORC_QKV: {
      int64_t q = m->n_q_heads, k = m->n_kv_heads, d = m->head_dim, qpg = q / k;
      if (tp <= k) {
        int64_t kpr = k / tp;
        if (m->qkv_order == 0) { s->nr[0] = kpr * (qpg + 2) * d; s->rb[0] = r * s->nr[0]; }
        else {
          s->nblk = 3;
          s->nr[0] = q / tp * d; s->rb[0] = r * s->nr[0];
          s->nr[1] = kpr * d;    s->rb[1] = q * d + r * s->nr[1];
          s->nr[2] = kpr * d;    s->rb[2] = (q + k) * d + r * s->nr[2];
        }
      } else {
        int64_t rep = tp / k, g = r / rep, j = r % rep, qpr = qpg / rep;
        if (m->qkv_order == 0) {
          int64_t base = g * (qpg + 2) * d;
          s->nblk = 2;
          s->nr[0] = qpr * d; s->rb[0] = base + j * qpr * d;
          s->nr[1] = 2 * d;   s->rb[1] = base + qpg * d;  s->rep[1] = (int32_t)rep;
        } else {
          s->nblk = 3;
          s->nr[0] = qpr * d; s->rb[0] = (int64_t)r * qpr * d;
          s->nr[1] = d;       s->rb[1] = q * d + g * d;        s->rep[1] = (int32_t)rep;
          s->nr[2] = d;       s->rb[2] = (q + k) * d + g * d;  s->rep[2] = (int32_t)rep;
        }
      }
      break;
    }
  }
  s->n = 0;
  for (int b = 0; b < s->nblk; b++) s->n += s->nr[b] * s->W;
}

/* local row i of a shard -> (block, row inside the block); blocks are stored one after the other */
static int orc_block_of(const orc_shard* q, int64_t i, int64_t* within) {
  int b = 0;
  while (b + 1 < q->nblk && i >= q->nr[b]) { i -= q->nr[b]; b++; }
  *within = i;
  return b;
}
/* first local row of block b */
static int64_t orc_block_start(const orc_shard* q, int b) {
  int64_t x = 0;
  for (int i = 0; i < b; i++) x += q->nr[i];
  return x;
}

void orc_layout_free(orc_layout* L) {
  if (!L) return;
  if (L->sh) for (int i = 0; i < L->c.pp * L->c.tp; i++) free(L->sh[i]);
  free(L->sh); free(L->n_sh); free(L->Lloc); free(L->lt); free(L->idx); free(L->tied_idx); free(L->failed); free(L);
}

/* Failure mask of an OLD layout ("Fault-tolerance through DP"; reading A26): failed[o] != 0 means
 * device o is lost with everything it held.  NULL clears the mask. */
void orc_layout_set_failed(orc_layout* L, const uint8_t* failed) {
  free(L->failed); L->failed = NULL;
  if (failed) {
    int n = L->c.tp * L->c.pp * L->c.dp;
    L->failed = (uint8_t*)malloc((size_t)n);
    for (int i = 0; i < n; i++) L->failed[i] = failed[i] ? 1 : 0;
  }
}
static int orc_is_failed(const orc_layout* L, int dev) { return L->failed && dev >= 0 && L->failed[dev]; }

int32_t orc_layout_new(const orc_model* m, const orc_cfg* c, orc_layout** out) {
  int rc = orc_validate(m, c);
  if (rc) return rc;
  if (!out) return ORC_ERR_ARG;
  orc_layout* L = (orc_layout*)calloc(1, sizeof(orc_layout));
  L->m = *m; L->c = *c;
  L->n_lt = orc_logical(m, c, NULL);
  L->lt = (orc_lt*)malloc(sizeof(orc_lt) * (size_t)L->n_lt);
  orc_logical(m, c, L->lt);
  int nsr = c->pp * c->tp;
  L->n_sh = (int32_t*)calloc((size_t)nsr, sizeof(int32_t));
  L->sh = (orc_shard**)calloc((size_t)nsr, sizeof(orc_shard*));
  L->Lloc = (int64_t*)calloc((size_t)nsr, sizeof(int64_t));
  L->idx = (int32_t*)malloc(sizeof(int32_t) * (size_t)c->pp * (size_t)L->n_lt);
  L->tied_idx = (int32_t*)malloc(sizeof(int32_t) * (size_t)c->pp);
  for (int i = 0; i < c->pp * L->n_lt; i++) L->idx[i] = -1;
  for (int i = 0; i < c->pp; i++) L->tied_idx[i] = -1;
  for (int s = 0; s < c->pp; s++) for (int r = 0; r < c->tp; r++) {
    int l_begin = orc_stage_begin(m->n_layers, c, s), l_end = orc_stage_begin(m->n_layers, c, s + 1);
    orc_shard* v = (orc_shard*)malloc(sizeof(orc_shard) * (size_t)(L->n_lt + 1));
    int k = 0; int64_t pos = 0;
    /* local order: pre tensors (stage 0), the stage's layers ascending, post tensors (last stage), tied replica */
    for (int pass = 0; pass < 3; pass++) for (int i = 0; i < L->n_lt; i++) {
      const orc_lt* t = &L->lt[i];
      if (t->where != pass) continue;
      if (pass == ORC_PRE && s != 0) continue;
      if (pass == ORC_LAYER && (t->layer < l_begin || t->layer >= l_end)) continue;
      if (pass == ORC_POST && s != c->pp - 1) continue;
      orc_make_shard(m, t, i, 0, c->tp, r, &v[k]); v[k].start = pos; pos += v[k].n;
      L->idx[s * L->n_lt + i] = k; k++;
    }
    if (m->tied && c->pp > 1 && s == c->pp - 1) {                  /* A11: replica of word_embeddings (tensor 0) */
      orc_make_shard(m, &L->lt[0], 0, 1, c->tp, r, &v[k]); v[k].start = pos; pos += v[k].n;
      L->tied_idx[s] = k; k++;
    }
    L->sh[s * c->tp + r] = v; L->n_sh[s * c->tp + r] = k; L->Lloc[s * c->tp + r] = pos;
  }
  *out = L;
  return ORC_OK;
}

int32_t orc_num_devices(const orc_layout* L) { return L->c.tp * L->c.pp * L->c.dp; }

/* device id = r + tp*(d + dp*s)  (A9: TP fastest, then DP, then PP) */
static void orc_coords(const orc_layout* L, int dev, int* d, int* s, int* r) {
  *r = dev % L->c.tp; *d = (dev / L->c.tp) % L->c.dp; *s = dev / (L->c.tp * L->c.dp);
}
static int orc_dev(const orc_layout* L, int d, int s, int r) { return r + L->c.tp * (d + L->c.dp * s); }

static int orc_dp_sharded(const orc_layout* L, int kind) {          /* A14 */
  return L->c.dist_opt && L->c.dp > 1 && kind >= 1;
}
static int orc_has_kind(const orc_layout* L, int kind) { return kind >= 0 && kind < 4 && ((L->m.kinds >> kind) & 1); }

/* flat range [lo,hi) of the (s,r) local space that buffer (d,s,r,kind) holds */
static void orc_flat_range(const orc_layout* L, int d, int s, int r, int kind, int64_t* lo, int64_t* hi) {
  int64_t n = L->Lloc[s * L->c.tp + r];
  if (!orc_has_kind(L, kind)) { *lo = 0; *hi = 0; return; }
  if (orc_dp_sharded(L, kind)) {
    /* A14: chunk = ceil(n / dp); A28: rounded up to a multiple of `align` elements: chunk = ceil(n / (dp*align)) * align */
    int64_t align = L->c.dist_opt_align > 1 ? L->c.dist_opt_align : 1;
    int64_t chunk = (n + (int64_t)L->c.dp * align - 1) / ((int64_t)L->c.dp * align) * align;
    int64_t a = (int64_t)d * chunk, b = (int64_t)(d + 1) * chunk;
    *lo = a < n ? a : n; *hi = b < n ? b : n;
  } else { *lo = 0; *hi = n; }
}

int64_t orc_buffer_elems(const orc_layout* L, int32_t dev, int32_t kind) {
  int d, s, r; int64_t lo, hi;
  orc_coords(L, dev, &d, &s, &r); orc_flat_range(L, d, s, r, kind, &lo, &hi);
  return hi - lo;
}

/* global_of: the l-th element of buffer (dev, kind) is element (row, col) of logical tensor lt */
int32_t orc_global_of(const orc_layout* L, int32_t dev, int32_t kind, int64_t l,
                      int32_t* lt, int32_t* post_copy, int64_t* row, int64_t* col) {
  int d, s, r; int64_t lo, hi;
  orc_coords(L, dev, &d, &s, &r); orc_flat_range(L, d, s, r, kind, &lo, &hi);
  if (l < 0 || l >= hi - lo) return ORC_ERR_ARG;
  int64_t g = lo + l;
  const orc_shard* v = L->sh[s * L->c.tp + r]; int n = L->n_sh[s * L->c.tp + r];
  int a = 0, b = n - 1;                        /* last shard with start <= g (empty shards cannot occur) */
  while (a < b) { int mid = (a + b + 1) / 2; if (v[mid].start <= g) a = mid; else b = mid - 1; }
  const orc_shard* q = &v[a];
  int64_t x = g - q->start, i = x / q->W, j = x % q->W;
  int64_t within; int blk = orc_block_of(q, i, &within);
  *lt = q->lt; *post_copy = q->post_copy; *row = q->rb[blk] + within; *col = q->c0 + j;
  return ORC_OK;
}

/* batch form of global_of for l in [l0, l0+count) */
int32_t orc_global_of_range(const orc_layout* L, int32_t dev, int32_t kind, int64_t l0, int64_t count,
                            int32_t* lt, int32_t* post_copy, int64_t* row, int64_t* col) {
  for (int64_t i = 0; i < count; i++) {
    int rc = orc_global_of(L, dev, kind, l0 + i, &lt[i], &post_copy[i], &row[i], &col[i]);
    if (rc) return rc;
  }
  return ORC_OK;
}

typedef struct { int32_t dev, d, s, r, post_copy; int64_t l; } orc_holder;

/* holders_of: every (device, local index) whose buffer of `kind` holds element (row, col) of tensor lt.
 * Returns the count; out must have room for 2*tp*dp entries. */
static int orc_holders(const orc_layout* L, int kind, int lt, int64_t row, int64_t col, orc_holder* out) {
  int n = 0;
  if (!orc_has_kind(L, kind)) return 0;
  for (int s = 0; s < L->c.pp; s++) for (int copy = 0; copy < 2; copy++) {
    int k = copy == 0 ? L->idx[s * L->n_lt + lt] : (lt == 0 ? L->tied_idx[s] : -1);
    if (k < 0) continue;                                   /* stage s does not hold this tensor (copy) */
    for (int r = 0; r < L->c.tp; r++) {
      const orc_shard* q = &L->sh[s * L->c.tp + r][k];
      if (col < q->c0 || col >= q->c0 + q->W) continue;
      int blk = -1;
      for (int b = 0; b < q->nblk; b++) if (row >= q->rb[b] && row < q->rb[b] + q->nr[b]) blk = b;
      if (blk < 0) continue;
      int64_t g = q->start + (orc_block_start(q, blk) + (row - q->rb[blk])) * q->W + (col - q->c0);
      for (int d = 0; d < L->c.dp; d++) {
        int64_t lo, hi; orc_flat_range(L, d, s, r, kind, &lo, &hi);
        if (g < lo || g >= hi) continue;
        out[n].dev = orc_dev(L, d, s, r); out[n].d = d; out[n].s = s; out[n].r = r;
        out[n].post_copy = q->post_copy; out[n].l = g - lo; n++;
      }
    }
  }
  return n;
}

int32_t orc_holders_of(const orc_layout* L, int32_t kind, int32_t lt, int64_t row, int64_t col,
                       int32_t cap, int32_t* dev, int64_t* l) {
  orc_holder* h = (orc_holder*)malloc(sizeof(orc_holder) * (size_t)(2 * L->c.tp * L->c.dp * L->c.pp + 2));
  int n = orc_holders(L, kind, lt, row, col, h);
  for (int i = 0; i < n && i < cap; i++) { dev[i] = h[i].dev; l[i] = h[i].l; }
  free(h);
  return n;
}

static int orc_same_model(const orc_layout* A, const orc_layout* B) {
  return memcmp(&A->m, &B->m, sizeof(orc_model)) == 0;
}

/* ---------------------------------------------------------------- cost matrix (A1-A5)
 * hold[o] = bytes old device o holds; need[n] = bytes new rank n needs;
 * overlap[n][o] = bytes of elements held by both (row-major [n_new][P], P = max(n_old, n_new)).
 * Element by element: each element of new rank n is looked up among the holders in the old layout.
 * only_layers != 0 restricts all three to transformer-layer tensors (for the paper's layer-only example P1). */
/* A26: a failed old device holds nothing: its column of the overlap matrix and its hold entry are zero. */
static void orc_drop_failed(const orc_layout* Lo, int nn, int P, int64_t* overlap, int64_t* hold) {
  int no = Lo->c.tp * Lo->c.pp * Lo->c.dp;
  for (int o = 0; o < no; o++) if (orc_is_failed(Lo, o)) {
    hold[o] = 0;
    for (int n = 0; n < nn; n++) overlap[(size_t)n * P + o] = 0;
  }
}

int32_t orc_overlap_elementwise(const orc_layout* Lo, const orc_layout* Ln, int32_t only_layers,
                                int64_t* overlap, int64_t* need, int64_t* hold) {
  if (!orc_same_model(Lo, Ln)) return ORC_ERR_ARG;
  int no = orc_num_devices(Lo), nn = orc_num_devices(Ln), P = no > nn ? no : nn;
  memset(overlap, 0, sizeof(int64_t) * (size_t)nn * (size_t)P);
  memset(need, 0, sizeof(int64_t) * (size_t)nn);
  memset(hold, 0, sizeof(int64_t) * (size_t)P);
  for (int o = 0; o < no; o++) for (int k = 0; k < 4; k++) {
    int64_t cnt = orc_buffer_elems(Lo, o, k), es = orc_elem_bytes(&Lo->m, k);
    if (!only_layers) { hold[o] += cnt * es; continue; }
    for (int64_t l = 0; l < cnt; l++) {
      int32_t lt, pc; int64_t row, col; orc_global_of(Lo, o, k, l, &lt, &pc, &row, &col);
      if (Lo->lt[lt].where == ORC_LAYER) hold[o] += es;
    }
  }
#pragma omp parallel for schedule(dynamic, 1)
  for (int n = 0; n < nn; n++) {
    orc_holder* h = (orc_holder*)malloc(sizeof(orc_holder) * (size_t)(2 * Lo->c.tp * Lo->c.dp * Lo->c.pp + 2));
    for (int k = 0; k < 4; k++) {
      int64_t cnt = orc_buffer_elems(Ln, n, k), es = orc_elem_bytes(&Ln->m, k);
      for (int64_t l = 0; l < cnt; l++) {
        int32_t lt, pc; int64_t row, col; orc_global_of(Ln, n, k, l, &lt, &pc, &row, &col);
        if (only_layers && Ln->lt[lt].where != ORC_LAYER) continue;
        need[n] += es;
        int nh = orc_holders(Lo, k, lt, row, col, h);
        for (int i = 0; i < nh; i++) {
          int dup = 0;                       /* a device holding the element twice counts once (cannot occur) */
          for (int j = 0; j < i; j++) if (h[j].dev == h[i].dev) dup = 1;
          if (!dup) overlap[(size_t)n * P + h[i].dev] += es;
        }
      }
    }
    free(h);
  }
  orc_drop_failed(Lo, nn, P, overlap, hold);
  return ORC_OK;
}

/* The paper's own treatment of DP ("DP Dimension"; reading A5): "we isolate the PP/TP processes
 * under different DP ranks.  If two processes have different DP ranks, even if their workloads on PP/TP are the same, we
 * regard the difference between the workloads to be infinite."  In the overlap form used here: a new rank and an old
 * device with different DP ranks share nothing that counts, so their cell is zero and the sketch never keeps bytes
 * local across DP groups.  Device id = r + tp*(d + dp*s) (A9).  Applied in place to overlap [n_new][P]. */
int32_t orc_mask_cross_dp(const orc_layout* Lo, const orc_layout* Ln, int64_t* overlap) {
  int no = orc_num_devices(Lo), nn = orc_num_devices(Ln), P = no > nn ? no : nn;
  for (int n = 0; n < nn; n++) {
    int dn, sn, rn; orc_coords(Ln, n, &dn, &sn, &rn);
    for (int o = 0; o < no; o++) {
      int dd, so, ro; orc_coords(Lo, o, &dd, &so, &ro);
      if (dd != dn) overlap[(size_t)n * P + o] = 0;
    }
  }
  return ORC_OK;
}

/* Second, separately written routine for layouts too large for element enumeration (config 5b): per pair of
 * tensor shards, count common elements row by row from the row/column ranges and the held flat ranges.
 * Validated against orc_overlap_elementwise on the tiny sweeps and on configs 1-2 (tests). */
static int64_t orc_isect(int64_t a0, int64_t a1, int64_t b0, int64_t b1) {
  int64_t lo = a0 > b0 ? a0 : b0, hi = a1 < b1 ? a1 : b1; return hi > lo ? hi - lo : 0;
}
/* columns [*c0,*c1) of logical row `row` that buffer range [lo,hi) of shard q holds; returns 0 if none */
static int orc_row_cols(const orc_shard* q, int64_t lo, int64_t hi, int64_t row, int64_t* c0, int64_t* c1) {
  for (int b = 0; b < q->nblk; b++) {
    if (row < q->rb[b] || row >= q->rb[b] + q->nr[b]) continue;
    int64_t g0 = q->start + (orc_block_start(q, b) + (row - q->rb[b])) * q->W, g1 = g0 + q->W;
    int64_t a = g0 > lo ? g0 : lo, e = g1 < hi ? g1 : hi;
    if (e <= a) return 0;
    *c0 = q->c0 + (a - g0); *c1 = q->c0 + (e - g0);
    return 1;
  }
  return 0;
}
int32_t orc_overlap_ranges(const orc_layout* Lo, const orc_layout* Ln, int64_t* overlap, int64_t* need,
                           int64_t* hold) {
  if (!orc_same_model(Lo, Ln)) return ORC_ERR_ARG;
  int no = orc_num_devices(Lo), nn = orc_num_devices(Ln), P = no > nn ? no : nn;
  memset(overlap, 0, sizeof(int64_t) * (size_t)nn * (size_t)P);
  memset(need, 0, sizeof(int64_t) * (size_t)nn);
  memset(hold, 0, sizeof(int64_t) * (size_t)P);
  for (int o = 0; o < no; o++) for (int k = 0; k < 4; k++) hold[o] += orc_buffer_elems(Lo, o, k) * orc_elem_bytes(&Lo->m, k);
  for (int n = 0; n < nn; n++) for (int k = 0; k < 4; k++) need[n] += orc_buffer_elems(Ln, n, k) * orc_elem_bytes(&Ln->m, k);
#pragma omp parallel for schedule(dynamic, 1)
  for (int n = 0; n < nn; n++) {
    int dn, sn, rn; orc_coords(Ln, n, &dn, &sn, &rn);
    const orc_shard* vn = Ln->sh[sn * Ln->c.tp + rn]; int cn = Ln->n_sh[sn * Ln->c.tp + rn];
    for (int o = 0; o < no; o++) {
      int dd, so, ro; orc_coords(Lo, o, &dd, &so, &ro);
      const orc_shard* vo = Lo->sh[so * Lo->c.tp + ro]; int co = Lo->n_sh[so * Lo->c.tp + ro];
      int64_t acc = 0;
      for (int k = 0; k < 4; k++) {
        int64_t nlo, nhi, olo, ohi, es = orc_elem_bytes(&Ln->m, k);
        orc_flat_range(Ln, dn, sn, rn, k, &nlo, &nhi); orc_flat_range(Lo, dd, so, ro, k, &olo, &ohi);
        if (nhi <= nlo || ohi <= olo) continue;
        for (int a = 0; a < cn; a++) for (int copy = 0; copy < 2; copy++) {
          const orc_shard* A = &vn[a];
          int b = copy == 0 ? Lo->idx[so * Lo->n_lt + A->lt] : (A->lt == 0 ? Lo->tied_idx[so] : -1);
          if (b < 0 || b >= co) continue;
          const orc_shard* B = &vo[b];
          int wholeA = nlo <= A->start && A->start + A->n <= nhi, wholeB = olo <= B->start && B->start + B->n <= ohi;
          if (orc_isect(A->start, A->start + A->n, nlo, nhi) == 0) continue;
          if (orc_isect(B->start, B->start + B->n, olo, ohi) == 0) continue;
          int64_t cols = orc_isect(A->c0, A->c0 + A->W, B->c0, B->c0 + B->W);
          if (!cols) continue;
          for (int ba = 0; ba < A->nblk; ba++) for (int bb = 0; bb < B->nblk; bb++) {
            int64_t r0 = A->rb[ba] > B->rb[bb] ? A->rb[ba] : B->rb[bb];
            int64_t r1a = A->rb[ba] + A->nr[ba], r1b = B->rb[bb] + B->nr[bb], r1 = r1a < r1b ? r1a : r1b;
            if (r1 <= r0) continue;
            if (wholeA && wholeB) { acc += (r1 - r0) * cols * es; continue; }
            for (int64_t row = r0; row < r1; row++) {            /* a held range cuts through rows: go row by row */
              int64_t a0, a1, b0, b1;
              if (!orc_row_cols(A, nlo, nhi, row, &a0, &a1)) continue;
              if (!orc_row_cols(B, olo, ohi, row, &b0, &b1)) continue;
              acc += orc_isect(a0, a1, b0, b1) * es;
            }
          }
        }
      }
      overlap[(size_t)n * P + o] = acc;
    }
  }
  orc_drop_failed(Lo, nn, P, overlap, hold);
  return ORC_OK;
}

/* ---------------------------------------------------------------- sketch (Eq. 1-4, Alg. 1; A4, A17, A18)
 * objective: local*(pi) = sum_n overlap[n][pi(n)], pi injective [0,n_new) -> [0,P), avail[p] != 0 (NULL = all). */
static void orc_bf_rec(const int64_t* ov, int nn, int P, const uint8_t* avail, int n, uint8_t* used, int32_t* cur,
                       int64_t acc, int64_t* best, int32_t* best_map, int64_t* count) {
  if (n == nn) {
    (*count)++;
    if (acc > *best) { *best = acc; memcpy(best_map, cur, sizeof(int32_t) * (size_t)nn); }
    return;
  }
  for (int p = 0; p < P; p++) {
    if (used[p] || (avail && !avail[p])) continue;
    used[p] = 1; cur[n] = p;
    orc_bf_rec(ov, nn, P, avail, n + 1, used, cur, acc + ov[(size_t)n * P + p], best, best_map, count);
    used[p] = 0;
  }
}
/* brute force over ALL injective maps; returns the number of maps tried (0 = infeasible) */
int64_t orc_sketch_bruteforce(const int64_t* overlap, int32_t n_new, int32_t P, const uint8_t* avail,
                              int32_t* best_map, int64_t* best_value) {
  uint8_t* used = (uint8_t*)calloc((size_t)P, 1); int32_t* cur = (int32_t*)calloc((size_t)n_new, sizeof(int32_t));
  int64_t best = -1, count = 0;
  orc_bf_rec(overlap, n_new, P, avail, 0, used, cur, 0, &best, best_map, &count);
  *best_value = best; free(used); free(cur);
  return count;
}

/* Algorithm 1: pad to k x k, Hungarian, drop padded pairs.  Padded rows are dummy new ranks that
 * overlap nothing (reading A4: maximise bytes staying local == minimise cost (BIG - overlap) with zero padding rows).
 * Plain O(k^3) Kuhn-Munkres with potentials on the minimisation form cost = maxv - overlap (unavailable: +inf). */
int32_t orc_sketch_hungarian(const int64_t* overlap, int32_t n_new, int32_t P, const uint8_t* avail,
                             int32_t* map, int64_t* value) {
  int k = P; if (n_new > P) return ORC_ERR_ARG;
  const int64_t INF = (int64_t)1 << 60;
  int64_t maxv = 0;
  for (int i = 0; i < n_new; i++) for (int j = 0; j < P; j++) if (overlap[(size_t)i * P + j] > maxv) maxv = overlap[(size_t)i * P + j];
  int64_t* u = (int64_t*)calloc((size_t)k + 1, 8); int64_t* v = (int64_t*)calloc((size_t)k + 1, 8);
  int* p = (int*)calloc((size_t)k + 1, sizeof(int)); int* way = (int*)calloc((size_t)k + 1, sizeof(int));
  int64_t* minv = (int64_t*)malloc(((size_t)k + 1) * 8); char* used = (char*)malloc((size_t)k + 1);
  int navail = 0; for (int j = 0; j < P; j++) if (!avail || avail[j]) navail++;
  if (navail < n_new) { free(u); free(v); free(p); free(way); free(minv); free(used); return ORC_ERR_ARG; }
#define COST(i, j) ((avail && !avail[(j)]) ? INF : ((i) < n_new ? maxv - overlap[(size_t)(i) * P + (j)] : (int64_t)0))
  for (int i = 1; i <= n_new; i++) {            /* padded rows (i > n_new) cost 0 everywhere: matching them is free */
    p[0] = i; int j0 = 0;
    for (int j = 0; j <= k; j++) { minv[j] = INF * 2; used[j] = 0; }
    do {
      used[j0] = 1; int i0 = p[j0], j1 = 0; int64_t delta = INF * 2;
      for (int j = 1; j <= k; j++) if (!used[j]) {
        int64_t cur = COST(i0 - 1, j - 1) - u[i0] - v[j];
        if (cur < minv[j]) { minv[j] = cur; way[j] = j0; }
        if (minv[j] < delta) { delta = minv[j]; j1 = j; }
      }
      for (int j = 0; j <= k; j++) if (used[j]) { u[p[j]] += delta; v[j] -= delta; } else minv[j] -= delta;
      j0 = j1;
    } while (p[j0] != 0);
    do { int j1 = way[j0]; p[j0] = p[j1]; j0 = j1; } while (j0);
  }
#undef COST
  int64_t tot = 0;
  for (int j = 1; j <= k; j++) if (p[j] >= 1 && p[j] <= n_new) { map[p[j] - 1] = j - 1; tot += overlap[(size_t)(p[j] - 1) * P + (j - 1)]; }
  *value = tot;
  free(u); free(v); free(p); free(way); free(minv); free(used);
  return ORC_OK;
}

/* ---------------------------------------------------------------- source rule (A6) and migration
 * New rank n = (d', s', r') placed on physical device p = device_map[n]; old logical rank j sits on physical j.
 *   (i)  local first: if old device p holds the element, the source is p (paper's Refer: stays in place);
 *   (ii) else the designated holder (d, s, r): s = the old stage holding the tensor (tied word_embeddings held by two
 *        stages: stage 0 for the `pre` copy, the last stage for the `post` copy); r = the unique TP rank holding it
 *        if the tensor is TP-sharded in old, else r' mod tp_old (in general: round-robin by r' over the ranks of that
 *        stage holding the element, A30); d = the unique DP rank whose flat range holds it if
 *        the kind is DP-sharded in old, else d' mod dp_old (round-robin over source groups). */
static int orc_pick_source(const orc_layout* Lo, const orc_layout* Ln, int n, int p, int kind,
                           int lt, int post_copy, int64_t row, int64_t col, orc_holder* h, orc_holder* src) {
  int nh = orc_holders(Lo, kind, lt, row, col, h);
  if (nh == 0) {
    /* reading A31: a padding row of the new layout's padded vocabulary that lies beyond the old layout's padded
     * vocabulary is held by no old device: it has no source and is zero-filled.  Anything else without a holder is
     * an error. */
    if (Lo->lt[lt].rows != Ln->lt[lt].rows && row >= Lo->lt[lt].rows && row < Ln->lt[lt].rows) return 2;
    return -1;
  }
  for (int i = 0; i < nh; i++) if (h[i].dev == p && !orc_is_failed(Lo, p)) { *src = h[i]; return 0; }   /* (i) */
  int dn, sn, rn; orc_coords(Ln, n, &dn, &sn, &rn);
  int smin = h[0].s, smax = h[0].s;
  for (int i = 1; i < nh; i++) { if (h[i].s < smin) smin = h[i].s; if (h[i].s > smax) smax = h[i].s; }
  int s_des = (smin == smax) ? smin : (post_copy ? smax : smin);
  int r_des = -1, d_first = -1, d_des;
  {
    /* the TP ranks of stage s_des holding the element, ascending: one if the element is TP-sharded, all tp if the
     * tensor is replicated, the tp/n_kv ranks of a KV group for a replicated K/V head (A30).  Round-robin over them
     * by the new TP rank: r = ranks[r' mod count]  (for a replicated tensor this is r' mod tp_old, A6) */
    int cnt = 0, last = -1;
    for (int i = 0; i < nh; i++) if (h[i].s == s_des && h[i].r != last) { last = h[i].r; cnt++; }
    int want = rn % cnt, seen = 0; last = -1;
    for (int i = 0; i < nh; i++) if (h[i].s == s_des && h[i].r != last) {
      last = h[i].r;
      if (seen == want) r_des = h[i].r;
      seen++;
    }
  }
  if (orc_dp_sharded(Lo, kind)) {
    for (int i = 0; i < nh; i++) if (h[i].s == s_des && h[i].r == r_des) d_first = h[i].d;
    d_des = d_first;
    if (orc_is_failed(Lo, orc_dev(Lo, d_des, s_des, r_des))) return -2;    /* A26: the only holder is lost */
  } else {
    /* A26: the designated DP rank, else the next surviving replica in cyclic DP order with the
     * same PP/TP ranks ("obtained from other DP groups via the PP/TP ranks") */
    d_des = -1;
    for (int j = 0; j < Lo->c.dp; j++) {
      int d = (dn % Lo->c.dp + j) % Lo->c.dp;
      if (!orc_is_failed(Lo, orc_dev(Lo, d, s_des, r_des))) { d_des = d; break; }
    }
    if (d_des < 0) return -2;                                              /* every replica is lost */
  }
  for (int i = 0; i < nh; i++) if (h[i].s == s_des && h[i].r == r_des && h[i].d == d_des) { *src = h[i]; return 1; }
  return -1;
}

/* source (old device, local index) of the elements l_list[i] of new buffer (n, kind) */
int32_t orc_source_of(const orc_layout* Lo, const orc_layout* Ln, const int32_t* device_map, int32_t n, int32_t kind,
                      const int64_t* l_list, int64_t count, int32_t* src_dev, int64_t* src_l) {
  orc_holder* h = (orc_holder*)malloc(sizeof(orc_holder) * (size_t)(2 * Lo->c.tp * Lo->c.dp * Lo->c.pp + 2));
  int rc = ORC_OK;
  for (int64_t i = 0; i < count; i++) {
    int32_t lt, pc; int64_t row, col; orc_holder s;
    if (orc_global_of(Ln, n, kind, l_list[i], &lt, &pc, &row, &col)) { rc = ORC_ERR_ARG; break; }
    int how = orc_pick_source(Lo, Ln, n, device_map[n], kind, lt, pc, row, col, h, &s);
    if (how < 0) { rc = how == -2 ? ORC_ERR_UNRECOVERABLE : ORC_ERR_ARG; break; }
    if (how == 2) { src_dev[i] = -1; src_l[i] = -1; continue; }      /* zero-filled: no source (A31) */
    src_dev[i] = s.dev; src_l[i] = s.l;
  }
  free(h);
  return rc;
}

static int orc_check_map(const int32_t* map, int nn, int P) {
  for (int i = 0; i < nn; i++) {
    if (map[i] < 0 || map[i] >= P) return ORC_ERR_ARG;
    for (int j = 0; j < i; j++) if (map[j] == map[i]) return ORC_ERR_ARG;
  }
  return ORC_OK;
}

/* Element-wise migration of local indices [l0, l1) of new buffer (n, kind):  dst[l] = src_bufs[o*4+kind][l'].
 * src_bufs: array [n_old*4] of host pointers; dst: the new buffer (n, kind) (NULL = count traffic only).
 * T (optional, [P][P] row-major, ADDED to): T[o][p] += elem bytes.  overrides (optional, ADDED to): number of
 * elements whose local-first source differs from the designated holder.  written (optional): per-element write
 * count of the destination buffer, incremented (pin P10).  fill (optional, ADDED to): bytes of this range that have
 * no source and are zero-filled (padding rows of a grown padded vocabulary, reading A31). */
int32_t orc_migrate_range_fill(const orc_layout* Lo, const orc_layout* Ln, const int32_t* device_map, int32_t n,
                               int32_t kind, int64_t l0, int64_t l1, const void* const* src_bufs, void* dst,
                               int64_t* T, int64_t* overrides, uint8_t* written, int64_t* fill);
int32_t orc_migrate_range(const orc_layout* Lo, const orc_layout* Ln, const int32_t* device_map, int32_t n,
                          int32_t kind, int64_t l0, int64_t l1, const void* const* src_bufs, void* dst,
                          int64_t* T, int64_t* overrides, uint8_t* written) {
  return orc_migrate_range_fill(Lo, Ln, device_map, n, kind, l0, l1, src_bufs, dst, T, overrides, written, NULL);
}
int32_t orc_migrate_range_fill(const orc_layout* Lo, const orc_layout* Ln, const int32_t* device_map, int32_t n,
                               int32_t kind, int64_t l0, int64_t l1, const void* const* src_bufs, void* dst,
                               int64_t* T, int64_t* overrides, uint8_t* written, int64_t* fill) {
  if (!orc_same_model(Lo, Ln)) return ORC_ERR_ARG;
  int no = orc_num_devices(Lo), nn = orc_num_devices(Ln), P = no > nn ? no : nn;
  if (orc_check_map(device_map, nn, P)) return ORC_ERR_ARG;
  int es = orc_elem_bytes(&Ln->m, kind), p = device_map[n];
  orc_holder* h = (orc_holder*)malloc(sizeof(orc_holder) * (size_t)(2 * Lo->c.tp * Lo->c.dp * Lo->c.pp + 2));
  int rc = ORC_OK;
  for (int64_t l = l0; l < l1; l++) {
    int32_t lt, pc; int64_t row, col; orc_holder s;
    if (orc_global_of(Ln, n, kind, l, &lt, &pc, &row, &col)) { rc = ORC_ERR_ARG; break; }
    int how = orc_pick_source(Lo, Ln, n, p, kind, lt, pc, row, col, h, &s);
    if (how < 0) { rc = how == -2 ? ORC_ERR_UNRECOVERABLE : ORC_ERR_ARG; break; }
    if (how == 2) {                          /* A31: no source, zero-fill; moves no bytes between devices */
      if (dst) memset((char*)dst + l * es, 0, (size_t)es);
      if (written) written[l]++;
      if (fill) *fill += es;
      continue;
    }
    if (dst) memcpy((char*)dst + l * es, (const char*)src_bufs[s.dev * 4 + kind] + s.l * es, (size_t)es);
    if (T) T[(size_t)s.dev * P + p] += es;
    if (written) written[l]++;
    if (overrides && how == 0) {             /* was the local source also the designated one? */
      orc_holder t; int save = p; (void)save;
      int how2 = orc_pick_source(Lo, Ln, n, -1, kind, lt, pc, row, col, h, &t);
      if (how2 >= 0 && t.dev != s.dev) (*overrides)++;
    }
  }
  free(h);
  return rc;
}

/* Whole migration: every (n, kind), all elements.  dst_bufs [n_new*4] may be NULL (traffic only). */
int32_t orc_migrate_fill(const orc_layout* Lo, const orc_layout* Ln, const int32_t* device_map,
                         const void* const* src_bufs, void* const* dst_bufs, int64_t* T, int64_t* overrides,
                         int64_t* fill);
int32_t orc_migrate(const orc_layout* Lo, const orc_layout* Ln, const int32_t* device_map,
                    const void* const* src_bufs, void* const* dst_bufs, int64_t* T, int64_t* overrides) {
  return orc_migrate_fill(Lo, Ln, device_map, src_bufs, dst_bufs, T, overrides, NULL);
}
/* fill (optional, [n_new], overwritten): bytes of each new rank that are zero-filled (reading A31) */
int32_t orc_migrate_fill(const orc_layout* Lo, const orc_layout* Ln, const int32_t* device_map,
                         const void* const* src_bufs, void* const* dst_bufs, int64_t* T, int64_t* overrides,
                         int64_t* fill) {
  int no = orc_num_devices(Lo), nn = orc_num_devices(Ln), P = no > nn ? no : nn;
  if (T) memset(T, 0, sizeof(int64_t) * (size_t)P * (size_t)P);
  if (overrides) *overrides = 0;
  if (fill) memset(fill, 0, sizeof(int64_t) * (size_t)nn);
  if (orc_check_map(device_map, nn, P)) return ORC_ERR_ARG;
  int rc_all = ORC_OK;
#pragma omp parallel for schedule(dynamic, 1)
  for (int n = 0; n < nn; n++) {
    /* T's column device_map[n] belongs to rank n alone (the map is injective): no two threads add to one cell */
    int64_t ovr = 0;
    for (int k = 0; k < 4; k++) {
      int64_t cnt = orc_buffer_elems(Ln, n, k);
      if (!cnt) continue;
      int rc = orc_migrate_range_fill(Lo, Ln, device_map, n, k, 0, cnt, src_bufs, dst_bufs ? dst_bufs[n * 4 + k] : NULL,
                                      T, overrides ? &ovr : NULL, NULL, fill ? &fill[n] : NULL);
      if (rc) {
#pragma omp critical
        rc_all = rc;
      }
    }
    if (overrides) {
#pragma omp atomic
      *overrides += ovr;
    }
  }
  return rc_all;
}

int32_t orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
