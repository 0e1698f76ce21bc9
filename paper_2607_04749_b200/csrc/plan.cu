// plan.cu — (a4) plan: turn (old layout, new layout, device_map) into the instruction lists of PAPER.md:193-201 as a
// table of 2-D strided copies ("slices"):
//   Refer  (workload in both prev and curr process)  -> local slice, old buffer -> new buffer on the same device
//   Send / Recv (workload moves)                      -> staged slice, packed into the contiguous segment of its
//                                                        (source, destination) pair — message coalescing
// Source of every needed element (reading A6): local first, else the designated holder.
//
// A (source device od, new rank n) unit is one cell of the traffic matrix and one pair segment; it is cut into sub-blocks
// of pieces, one warp each.  Three launches: pass 1 counts slices / chunks / bytes per sub-block (no atomics); a
// single-CTA scan sums the sub-blocks of each unit and turns the unit counts into slice indices, chunk indices and segment
// offsets (warp-shuffle prefix sums); pass 2 recomputes the slices, writes them at their final positions and expands them
// into copy work items ("chunks") warp-cooperatively.  Order inside a segment is canonical (piece order), so the staging
// layout is deterministic.
#include <algorithm>
#include <cstring>
#include <vector>
#include "etc_internal.h"
#include "plan_types.h"

bool etc_same_model(const etc_layout* a, const etc_layout* b);

namespace etc {

struct Rect { int32_t r0, nr, c0, nc; };

__device__ __forceinline__ bool rect_isect(const Piece& a, const Piece& b, Rect& out) {
  const int r0 = max(a.r0, b.r0), r1 = min(a.r0 + a.nr, b.r0 + b.nr);
  const int c0 = max(a.c0, b.c0), c1 = min(a.c0 + a.nc, b.c0 + b.nc);
  out = Rect{r0, r1 - r0, c0, c1 - c0};
  return r1 > r0 && c1 > c0;
}

// Is old piece o the designated holder for new piece q (reading A6 (ii))?  With a failure mask (reading A26,
// PAPER.md:173-177) the designated DP rank is the first SURVIVING replica in cyclic DP order starting at d' mod dp_old,
// with the same PP/TP ranks; the caller has already skipped pieces of failed devices.
__device__ __forceinline__ bool designated(const Piece& o, const Piece& q, int tp_old, int dp_old,
                                           const uint8_t* __restrict__ failed) {
  const bool stage_ok = (o.flags & PF_SOLE_INST) || ((o.flags & PF_POST_COPY) == (q.flags & PF_POST_COPY));
  const bool r_ok = o.r == o.rbase + q.r % o.rep;      // round-robin by r' over the TP ranks holding it (A6, A30)
  if (!(stage_ok && r_ok)) return false;
  if (o.flags & PF_DP_SHARDED) return true;
  int d_des = q.d % dp_old;
  if (failed) {
    int j = 0;
    for (; j < dp_old; ++j) {
      const int d = (d_des + j) % dp_old;
      if (!failed[o.r + tp_old * (d + dp_old * o.s)]) { d_des = d; break; }
    }
    if (j == dp_old) return false;
  }
  return o.d == d_des;
}

// I minus the flat interval [b0,b1) of the shard (row pitch W) that I lives in.  I's first element is local
// (i0, j0).  Writes up to 4 rectangles (logical coordinates) and returns how many.
__device__ __forceinline__ int subtract_interval(const Rect& I, int64_t i0, int64_t j0, int64_t W, int64_t b0, int64_t b1,
                                                 Rect out[4]) {
  if (b1 <= b0) { out[0] = I; return 1; }
  const int64_t i1 = i0 + I.nr, j1 = j0 + I.nc;
  const int64_t ib = b0 / W, jb = b0 - ib * W, ie = b1 / W, je = b1 - ie * W;
  int n = 0;
  // A: rows strictly above the interval's first row
  { const int64_t e = min(i1, ib); if (e > i0) out[n++] = Rect{I.r0, (int32_t)(e - i0), I.c0, I.nc}; }
  // B: the interval's first row, columns before it starts
  if (ib >= i0 && ib < i1) { const int64_t e = min(j1, jb); if (e > j0) out[n++] = Rect{(int32_t)(I.r0 + (ib - i0)), 1, I.c0, (int32_t)(e - j0)}; }
  // C: the interval's last (partial) row, columns after it ends
  if (ie >= i0 && ie < i1) { const int64_t s = max(j0, je); if (j1 > s) out[n++] = Rect{(int32_t)(I.r0 + (ie - i0)), 1, (int32_t)(I.c0 + (s - j0)), (int32_t)(j1 - s)}; }
  // D: rows strictly below the interval's last row
  { const int64_t s = max(i0, ie + 1); if (i1 > s) out[n++] = Rect{(int32_t)(I.r0 + (s - i0)), (int32_t)(i1 - s), I.c0, I.nc}; }
  return n;
}

struct SliceGeom {           // one 2-D strided copy
  int64_t src_off, dst_off, row_bytes;
  int32_t src_stride, dst_stride, nrows, kind;
};

__device__ __forceinline__ SliceGeom make_slice(const Rect& R, const Piece& o, const Piece& q, int es, int kind) {
  SliceGeom s;
  s.src_off = o.boff + ((int64_t)(R.r0 - o.r0) * o.W + (R.c0 - o.c0)) * es;
  s.dst_off = q.boff + ((int64_t)(R.r0 - q.r0) * q.W + (R.c0 - q.c0)) * es;
  s.src_stride = o.W * es; s.dst_stride = q.W * es;
  s.nrows = R.nr; s.row_bytes = (int64_t)R.nc * es; s.kind = kind;
  if (s.nrows > 1 && s.row_bytes == s.src_stride && s.row_bytes == s.dst_stride) {   // contiguous on both sides
    s.row_bytes *= s.nrows; s.nrows = 1;
  }
  return s;
}

// widest power-of-two access (<= 16 bytes) that every address of a slice is aligned to.  Staging offsets of slices are
// multiples of 16 and the staging pitch is row_bytes, so the staging side adds nothing.
__device__ __forceinline__ int vec_of(int64_t a) {
  const int64_t low = a & -a;
  return a == 0 ? 16 : (low >= 16 ? 16 : (int)low);
}
__device__ __forceinline__ int slice_vec(int64_t src_off, int64_t dst_off, int64_t row_bytes, int32_t src_stride,
                                         int32_t dst_stride, int32_t nrows) {
  int64_t al = src_off | dst_off | row_bytes;
  if (nrows > 1) al |= (int64_t)src_stride | (int64_t)dst_stride;
  return vec_of(al);
}
__device__ __forceinline__ int64_t slice_chunks(const SliceGeom& s) {
  if (s.nrows == 1) return (s.row_bytes + ETC_CHUNK_BYTES - 1) / ETC_CHUNK_BYTES;
  if (s.row_bytes >= ETC_CHUNK_BYTES) return (int64_t)s.nrows * ((s.row_bytes + ETC_CHUNK_BYTES - 1) / ETC_CHUNK_BYTES);
  const int rpc = rows_per_chunk(s.row_bytes, slice_vec(s.src_off, s.dst_off, s.row_bytes, s.src_stride, s.dst_stride, s.nrows) == 16);
  return (s.nrows + rpc - 1) / rpc;
}
__device__ __forceinline__ int64_t slice_padded(const SliceGeom& s) { return (s.nrows * s.row_bytes + 15) & ~(int64_t)15; }

// Enumerate, in canonical order, the slices that new piece q receives from source device od.
template <typename F>
__device__ __forceinline__ void for_each_slice(const DeviceTables& oldT, const Piece& q, int od, int p, bool local_unit,
                                               int es, int kind, const uint8_t* __restrict__ failed, F&& f) {
  if (failed && failed[od]) return;                                              // a failed device sources nothing
  int j = oldT.first[(size_t)od * oldT.n_grp + q.grp];
  if (j < 0) return;
  const int oe = oldT.dev_start[od + 1];
  for (; j < oe; ++j) {
    const Piece o = oldT.pieces[j];
    if (o.grp != q.grp) break;
    Rect I;
    if (!rect_isect(q, o, I)) continue;
    if (local_unit) { f(make_slice(I, o, q, es, kind)); continue; }              // (i) local first
    if (!designated(o, q, oldT.tp, oldT.dp, failed)) continue;                   // (ii) designated holder only
    Rect parts[4]; int np = 1; parts[0] = I;
    if (p >= 0 && p < oldT.n_dev && !(failed && failed[p])) {                    // minus what the destination device holds
      const int pj = oldT.first[(size_t)p * oldT.n_grp + q.grp];
      if (pj >= 0) {
        const Piece& h = oldT.pieces[pj];
        // p holds these elements only if its TP rank is one of those holding them; all such ranks store them at the
        // same shard-local position (same shard, or the K/V block of one KV group, A30): subtract p's held flat range
        if (h.r >= o.rbase && h.r < o.rbase + o.rep)
          np = subtract_interval(I, (int64_t)o.lrow0 + (I.r0 - o.r0), (int64_t)o.lcol0 + (I.c0 - o.c0), o.W, h.f0, h.f1, parts);
      }
    }
    for (int k = 0; k < np; ++k) f(make_slice(parts[k], o, q, es, kind));
  }
}

__device__ __forceinline__ int64_t warp_sum64(int64_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ int64_t warp_excl_scan64(int64_t v, int lane, int64_t& total) {
  int64_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int64_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  total = __shfl_sync(0xffffffffu, x, 31);
  return x - v;
}

constexpr int PLAN_WARPS = 8;

// A unit u = (kq * n_old + od) * n_new + n (kq = 0 unless the plan is kind-major: then kq = state kind) is cut into B
// sub-blocks of `span` consecutive pieces of rank n (span a multiple of 32), one warp each, so that small device counts
// still fill the machine.  [i0,i1) = the piece range of sub-block b.
__device__ __forceinline__ void sub_range(const DeviceTables& newT, int n, int kq, int K, int B, int b, int& i0, int& i1) {
  const int qb = K == 1 ? newT.dev_start[n] : newT.kind_start[n * (ETC_NUM_KINDS + 1) + kq];
  const int qe = K == 1 ? newT.dev_start[n + 1] : newT.kind_start[n * (ETC_NUM_KINDS + 1) + kq + 1];
  const int span = (((qe - qb) + B - 1) / B + 31) & ~31;
  i0 = min(qe, qb + b * span); i1 = min(qe, i0 + span);
}

// pass 1: per-(unit, sub-block) counts.
__global__ void __launch_bounds__(PLAN_WARPS * 32)
plan_count_kernel(DeviceTables oldT, DeviceTables newT, const int32_t* __restrict__ device_map,
                  const uint8_t* __restrict__ failed, int K, int B, BlockCount* __restrict__ blocks) {
  const int lane = threadIdx.x & 31;
  const long long w = (long long)blockIdx.x * PLAN_WARPS + (threadIdx.x >> 5);
  const long long U = (long long)K * oldT.n_dev * newT.n_dev;
  if (w >= U * B) return;
  const long long u = w / B; const int b = (int)(w % B);
  const int n = (int)(u % newT.n_dev), od = (int)((u / newT.n_dev) % oldT.n_dev), kq = (int)(u / newT.n_dev / oldT.n_dev);
  const int p = device_map[n];
  const bool local_unit = (od == p);
  int64_t n_sl = 0, n_ch = 0, bytes = 0, padded = 0;
  bool common = false;
  for (int k = lane; k < newT.mask_words; k += 32)
    common |= (newT.ltmask[(size_t)n * newT.mask_words + k] & oldT.ltmask[(size_t)od * oldT.mask_words + k]) != 0;
  if (__any_sync(0xffffffffu, common)) {
    int i0, i1; sub_range(newT, n, kq, K, B, b, i0, i1);
    for (int i = i0 + lane; i < i1; i += 32) {
      const Piece q = newT.pieces[i];
      const int kind = q.grp / newT.n_tensors, es = newT.elem_bytes[kind];
      for_each_slice(oldT, q, od, p, local_unit, es, kind, failed, [&](const SliceGeom& s) {
        n_sl += 1; n_ch += slice_chunks(s); bytes += s.nrows * s.row_bytes; padded += slice_padded(s);
      });
    }
  }
  n_sl = warp_sum64(n_sl); n_ch = warp_sum64(n_ch); bytes = warp_sum64(bytes); padded = warp_sum64(padded);
  if (lane == 0) blocks[w] = BlockCount{n_sl, n_ch, padded, bytes};
}

// single-CTA exclusive scan over units (+ map validation, traffic matrix, totals)
constexpr int SCAN_THREADS = 1024;
__global__ void __launch_bounds__(SCAN_THREADS)
plan_scan_kernel(const BlockCount* __restrict__ blocks, int B, long long U, int K, int n_old, int n_new, int P, int flags,
                 const int32_t* __restrict__ device_map, int32_t* __restrict__ map_copy, UnitBase* __restrict__ bases,
                 int64_t* __restrict__ traffic, PlanTotals* __restrict__ totals, PlanTotals* __restrict__ totals_host,
                 int64_t bound_slices, int64_t bound_chunks, int64_t bound_staging) {
  __shared__ int64_t s_w[5][32];
  __shared__ int64_t s_carry[5];
  __shared__ int64_t s_loc[32], s_rem[32];
  __shared__ uint32_t s_seen[1024];          // P <= 32767 bits
  __shared__ int s_bad;
  __shared__ int64_t s_kind[ETC_NUM_KINDS][3];
  const long long U1 = U / K;                                  // units per kind (kind-major) or all units
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid < ETC_NUM_KINDS * 3) s_kind[tid / 3][tid % 3] = 0;
  if (tid < 5) s_carry[tid] = 0;
  if (tid == 0) s_bad = 0;
  for (int i = tid; i < 1024; i += SCAN_THREADS) s_seen[i] = 0;
  __syncthreads();
  for (int n = tid; n < n_new; n += SCAN_THREADS) {            // injective into [0,P)?  (and the plan keeps its own copy)
    const int p = device_map[n];
    if (map_copy != device_map) map_copy[n] = p;
    if (p < 0 || p >= P) s_bad = 1;
    else if (atomicOr(&s_seen[p >> 5], 1u << (p & 31)) & (1u << (p & 31))) s_bad = 1;
  }
  for (long long i = tid; i < (long long)P * P; i += SCAN_THREADS) traffic[i] = 0;
  __syncthreads();
  const bool bad = s_bad != 0;
  int64_t loc = 0, rem = 0;
  for (long long base = 0; base < U; base += SCAN_THREADS) {
    const long long u = base + tid;
    BlockCount c{0, 0, 0, 0};
    bool staged = false; int od = 0, p = 0;
    if (u < U) {
      for (int k = 0; k < B; ++k) {                             // the unit's sub-blocks
        const BlockCount x = blocks[u * B + k];
        c.slices += x.slices; c.chunks += x.chunks; c.padded += x.padded; c.bytes += x.bytes;
      }
      od = (int)((u / n_new) % n_old); p = device_map[(int)(u % n_new)];
      staged = !(flags & ETC_ALL_DIRECT) && ((od != p) || (flags & ETC_ALL_STAGED));
      c.padded = (c.padded + 511) & ~(int64_t)511;             // pair segments start 512-byte aligned
    }
    int64_t v[5];
    v[0] = staged ? c.slices : 0; v[1] = staged ? c.chunks : 0; v[2] = staged ? c.padded : 0;
    v[3] = staged ? 0 : c.slices; v[4] = staged ? 0 : c.chunks;
    int64_t ex[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) { int64_t tot; ex[k] = warp_excl_scan64(v[k], lane, tot); if (lane == 31) s_w[k][wid] = tot; }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
      for (int k = 0; k < 5; ++k) { int64_t tot; s_w[k][lane] = warp_excl_scan64(s_w[k][lane], lane, tot); }
    }
    __syncthreads();
    if (u < U) {
      UnitBase ub;
      ub.slice0 = s_carry[staged ? 0 : 3] + s_w[staged ? 0 : 3][wid] + ex[staged ? 0 : 3];
      ub.chunk0 = s_carry[staged ? 1 : 4] + s_w[staged ? 1 : 4][wid] + ex[staged ? 1 : 4];
      ub.stg0 = staged ? s_carry[2] + s_w[2][wid] + ex[2] : -1;
      bases[u] = ub;
      if (K > 1 && u % U1 == 0) {                              // first unit of a kind: where the kind's tables start
        const int kq = (int)(u / U1);
        s_kind[kq][0] = s_carry[1] + s_w[1][wid] + ex[1];
        s_kind[kq][1] = s_carry[2] + s_w[2][wid] + ex[2];
        s_kind[kq][2] = s_carry[4] + s_w[4][wid] + ex[4];
      }
      if (!bad && c.bytes) {
        atomicAdd(reinterpret_cast<unsigned long long*>(&traffic[(size_t)od * P + p]), (unsigned long long)c.bytes);
        if (od == p) loc += c.bytes; else rem += c.bytes;
      }
    }
    __syncthreads();
    if (tid == SCAN_THREADS - 1) {
#pragma unroll
      for (int k = 0; k < 5; ++k) s_carry[k] += s_w[k][wid] + ex[k] + v[k];
    }
    __syncthreads();
  }
  loc = warp_sum64(loc); rem = warp_sum64(rem);
  if (lane == 0) { s_loc[wid] = loc; s_rem[wid] = rem; }
  __syncthreads();
  if (wid == 0) {
    loc = warp_sum64(s_loc[lane]); rem = warp_sum64(s_rem[lane]);
    if (lane == 0) {
      PlanTotals t;
      t.n_slices_staged = s_carry[0]; t.n_chunks_staged = s_carry[1]; t.staging_bytes = s_carry[2];
      t.n_slices_local = s_carry[3]; t.n_chunks_local = s_carry[4];
      t.local_bytes = loc; t.remote_bytes = rem; t.bad_map = bad ? 1 : 0;
      t.fill_bytes = 0; t.n_fills = 0;                          // plan_fills_kernel adds to these
      // ETC_NO_SYNC: the tables were sized from host-side upper bounds before these counts existed.  Should a bound
      // ever fall short, or the map be bad, the counts are zeroed so that no later kernel writes or copies anything.
      t.overflow = (bound_slices > 0 && (t.n_slices_staged > bound_slices || t.n_slices_local > bound_slices ||
                                         t.n_chunks_staged + t.n_chunks_local > bound_chunks ||   // grids, the ordered
                                         t.staging_bytes > bound_staging)) ? 1 : 0;                 // lists and ranks hold the SUM
      if (bound_slices > 0 && (t.overflow || t.bad_map)) {
        t.n_slices_staged = t.n_chunks_staged = t.n_slices_local = t.n_chunks_local = 0; t.staging_bytes = 0;
      }
      for (int k = 0; k < ETC_NUM_KINDS; ++k) for (int j = 0; j < 3; ++j) t.kind_base[k][j] = s_kind[k][j];
      t.kind_base[ETC_NUM_KINDS][0] = s_carry[1]; t.kind_base[ETC_NUM_KINDS][1] = s_carry[2];
      t.kind_base[ETC_NUM_KINDS][2] = s_carry[4];
      *totals = t;
      if (totals_host) *totals_host = t;                        // pinned host slot: the sizes the host is waiting for
    }
  }
}

// The copy work items of one slice (see slice_chunks for the count).  Built once per slice — the divisions that depend on
// the slice alone (rows per chunk, chunks per row) are done here, not once per chunk: a unit that keeps a whole
// embedding shard local is a single slice of thousands of chunks, expanded by one warp.
struct ChunkCutter {
  Chunk proto;                 // fields every chunk of the slice shares
  int64_t src_off, dst_off, stg_off, row_bytes;
  int32_t src_stride, dst_stride, nrows;
  uint32_t cpr;                // chunks per row (rows >= ETC_CHUNK_BYTES, or one contiguous run)
  int rpc;                     // rows per chunk (shorter rows)
  bool long_rows;
  __device__ __forceinline__ ChunkCutter() {}
  // the cutter that lane `from` holds, in every lane of the warp
  __device__ __forceinline__ ChunkCutter bcast(int from) const {
    const unsigned m = 0xffffffffu;
    ChunkCutter c;
    c.proto.src_buf = (uint16_t)__shfl_sync(m, (int)proto.src_buf, from); c.proto.dst_buf = (uint16_t)__shfl_sync(m, (int)proto.dst_buf, from);
    c.proto.vec = (int16_t)__shfl_sync(m, (int)proto.vec, from); c.proto.pad = 0;
    c.src_off = __shfl_sync(m, (long long)src_off, from); c.dst_off = __shfl_sync(m, (long long)dst_off, from);
    c.stg_off = __shfl_sync(m, (long long)stg_off, from); c.row_bytes = __shfl_sync(m, (long long)row_bytes, from);
    c.src_stride = __shfl_sync(m, src_stride, from); c.dst_stride = __shfl_sync(m, dst_stride, from);
    c.proto.src_stride = c.src_stride; c.proto.dst_stride = c.dst_stride;
    c.nrows = __shfl_sync(m, nrows, from); c.cpr = __shfl_sync(m, cpr, from); c.rpc = __shfl_sync(m, rpc, from);
    c.long_rows = __shfl_sync(m, (int)long_rows, from) != 0;
    return c;
  }
  __device__ __forceinline__ ChunkCutter(const etc_slice& s, int vec) {
    proto.src_buf = (uint16_t)(s.src_dev * ETC_NUM_KINDS + s.kind); proto.dst_buf = (uint16_t)(s.dst_rank * ETC_NUM_KINDS + s.kind);
    proto.src_stride = s.src_stride; proto.dst_stride = s.dst_stride; proto.pad = 0; proto.vec = (int16_t)vec;
    src_off = s.src_off; dst_off = s.dst_off; stg_off = s.stg_off >= 0 ? s.stg_off : 0; row_bytes = s.row_bytes;
    src_stride = s.src_stride; dst_stride = s.dst_stride; nrows = s.nrows;
    long_rows = s.nrows == 1 || s.row_bytes >= ETC_CHUNK_BYTES;
    cpr = (uint32_t)((s.row_bytes + ETC_CHUNK_BYTES - 1) / ETC_CHUNK_BYTES);
    rpc = long_rows ? 1 : rows_per_chunk(s.row_bytes, vec == 16);
  }
  __device__ __forceinline__ Chunk cut(long long k) const {
    Chunk ch = proto;
    if (long_rows) {
      long long row = 0; uint32_t part = (uint32_t)k;            // a single row: chunk k is its k-th part
      if (nrows != 1) { row = k / cpr; part = (uint32_t)(k - row * cpr); }
      const int64_t b = (int64_t)part * ETC_CHUNK_BYTES;
      ch.src_off = src_off + row * src_stride + b;
      ch.dst_off = dst_off + row * dst_stride + b;
      ch.stg_off = stg_off + row * row_bytes + b;
      ch.nrows = 1; ch.row_bytes = (int32_t)min((int64_t)ETC_CHUNK_BYTES, row_bytes - b);
    } else {
      const long long row = k * rpc;
      ch.src_off = src_off + row * src_stride;
      ch.dst_off = dst_off + row * dst_stride;
      ch.stg_off = stg_off + row * row_bytes;
      ch.nrows = (int32_t)min((long long)rpc, nrows - row); ch.row_bytes = (int32_t)row_bytes;
    }
    return ch;
  }
};

// pass 2: recompute the slices of each (unit, sub-block), write the slice records at their final positions — unit base
// (scan) + earlier sub-blocks of the unit + warp-level prefix inside the sub-block — and expand them into chunks: the
// warp walks over the slices its lanes have just written and the 32 lanes cut chunk k, k + 32, ... of each.
__global__ void __launch_bounds__(PLAN_WARPS * 32)
plan_fill_kernel(DeviceTables oldT, DeviceTables newT, const int32_t* __restrict__ device_map,
                 const uint8_t* __restrict__ failed, int flags, int K, int B,
                 const BlockCount* __restrict__ blocks, const UnitBase* __restrict__ bases,
                 etc_slice* __restrict__ sl_staged, etc_slice* __restrict__ sl_local,
                 Chunk* __restrict__ ch_staged, Chunk* __restrict__ ch_local, const PlanTotals* __restrict__ lazy) {
  if (lazy && (lazy->bad_map || lazy->overflow)) return;
  const int lane = threadIdx.x & 31;
  const long long w = (long long)blockIdx.x * PLAN_WARPS + (threadIdx.x >> 5);
  const long long U = (long long)K * oldT.n_dev * newT.n_dev;
  if (w >= U * B) return;
  const long long u = w / B; const int b = (int)(w % B);
  if (blocks[w].slices == 0) return;
  const UnitBase ub = bases[u];
  const int n = (int)(u % newT.n_dev), od = (int)((u / newT.n_dev) % oldT.n_dev), kq = (int)(u / newT.n_dev / oldT.n_dev);
  const int p = device_map[n];
  const bool local_unit = (od == p), staged = !(flags & ETC_ALL_DIRECT) && (!local_unit || (flags & ETC_ALL_STAGED));
  etc_slice* sl_out = staged ? sl_staged : sl_local;
  Chunk* ch_out = staged ? ch_staged : ch_local;
  int64_t pre_sl = 0, pre_ch = 0, pre_pad = 0;                 // totals of the unit's earlier sub-blocks
  for (int k = lane; k < b; k += 32) { const BlockCount c = blocks[u * B + k]; pre_sl += c.slices; pre_ch += c.chunks; pre_pad += c.padded; }
  int64_t run_sl = ub.slice0 + warp_sum64(pre_sl), run_ch = ub.chunk0 + warp_sum64(pre_ch);
  int64_t run_stg = (staged ? ub.stg0 : 0) + warp_sum64(pre_pad);
  int i0, i1; sub_range(newT, n, kq, K, B, b, i0, i1);
  for (int ib = i0; ib < i1; ib += 32) {                       // all lanes iterate together (warp scans inside)
    const int i = ib + lane;
    Piece q; int kind = 0, es = 0;
    int64_t my_sl = 0, my_ch = 0, my_pad = 0;
    if (i < i1) {
      q = newT.pieces[i]; kind = q.grp / newT.n_tensors; es = newT.elem_bytes[kind];
      for_each_slice(oldT, q, od, p, local_unit, es, kind, failed, [&](const SliceGeom& s) {
        my_sl += 1; my_ch += slice_chunks(s); my_pad += slice_padded(s);
      });
    }
    int64_t tot_sl, tot_ch, tot_pad;
    int64_t o_sl = run_sl + warp_excl_scan64(my_sl, lane, tot_sl);       // warp-level prefix sums for slice offsets
    int64_t o_ch = run_ch + warp_excl_scan64(my_ch, lane, tot_ch);
    int64_t o_stg = run_stg + warp_excl_scan64(my_pad, lane, tot_pad);
    if (i < i1 && my_sl) {
      for_each_slice(oldT, q, od, p, local_unit, es, kind, failed, [&](const SliceGeom& s) {
        etc_slice r;
        r.src_off = s.src_off; r.dst_off = s.dst_off; r.stg_off = staged ? o_stg : -1; r.row_bytes = s.row_bytes;
        r.src_stride = s.src_stride; r.dst_stride = s.dst_stride; r.nrows = s.nrows;
        r.src_dev = od; r.dst_rank = n; r.dst_phys = p; r.kind = kind; r.pad = 0;
        sl_out[o_sl] = r;
        o_sl += 1; o_stg += slice_padded(s);
      });
    }
    // chunk expansion of the slices [run_sl, run_sl + tot_sl) this iteration wrote, whose chunks are
    // [run_ch, run_ch + tot_ch) in the same order
    // 32 slices at a time: every lane reads ONE of the records (written by a lane of this warp just above) and works out
    // its chunk count and cutter — the divisions of 32 slices side by side — then the warp takes the slices in turn,
    // the cutter handed round by shuffles, and the 32 lanes cut chunk k, k + 32, ... of it
    __syncwarp();
    int64_t c0 = run_ch;
    for (int64_t jb = 0; jb < tot_sl; jb += 32) {
      const int nb = (int)min((int64_t)32, tot_sl - jb);
      ChunkCutter mine; long long my_n = 0;
      if (lane < nb) {
        const etc_slice s = sl_out[run_sl + jb + lane];
        const int vec = slice_vec(s.src_off, s.dst_off, s.row_bytes, s.src_stride, s.dst_stride, s.nrows);
        SliceGeom g; g.src_off = s.src_off; g.dst_off = s.dst_off; g.row_bytes = s.row_bytes; g.src_stride = s.src_stride;
        g.dst_stride = s.dst_stride; g.nrows = s.nrows; g.kind = s.kind;
        my_n = slice_chunks(g);
        mine = ChunkCutter(s, vec);
      } else {
        mine = ChunkCutter(etc_slice{0, 0, 0, 16, 16, 16, 1, 0, 0, 0, 0, 0}, 16);   // unused filler with defined fields
      }
      for (int j = 0; j < nb; ++j) {
        const long long nch = __shfl_sync(0xffffffffu, my_n, j);
        const ChunkCutter cutter = mine.bcast(j);
        for (long long k = lane; k < nch; k += 32) ch_out[c0 + k] = cutter.cut(k);
        c0 += nch;
      }
    }
    run_sl += tot_sl; run_ch += tot_ch; run_stg += tot_pad;
  }
}

// Zero-fill list (reading A31): a row of an embedding tensor of the new layout that lies beyond the old layout's padded
// vocabulary (rows >= old_rows) is held by no old device.  One thread per new piece; a piece's rows beyond old_rows are
// one descriptor (an etc_slice with no source).  Runs only when the padded vocabulary grew.
__global__ void __launch_bounds__(256)
plan_fills_kernel(DeviceTables newT, const int32_t* __restrict__ device_map, int old_rows, int lm_head_id,
                  etc_slice* __restrict__ fills, PlanTotals* __restrict__ totals) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= newT.n_pieces) return;
  // plan_scan_kernel ran before this kernel on the same stream: a plan it found unusable (bad map, bound overflow) must
  // write nothing at all, so it gets no zero-fill descriptors either (n_fills stays 0 and migrate_fill_kernel leaves)
  if (totals->bad_map || totals->overflow) return;
  const Piece q = newT.pieces[i];
  const int t = q.grp % newT.n_tensors, kind = q.grp / newT.n_tensors;
  if (t != 0 && t != lm_head_id) return;
  const int r0 = max(q.r0, old_rows), r1 = q.r0 + q.nr;
  if (r1 <= r0) return;
  const int es = newT.elem_bytes[kind];
  etc_slice f;
  f.src_off = -1; f.stg_off = -1; f.src_stride = 0; f.src_dev = -1; f.pad = 0;
  f.dst_off = q.boff + (int64_t)(r0 - q.r0) * q.W * es;
  f.row_bytes = (int64_t)q.nc * es; f.dst_stride = q.W * es; f.nrows = r1 - r0;
  if (f.nrows > 1 && f.row_bytes == f.dst_stride && f.row_bytes * f.nrows < (1ll << 31)) { f.row_bytes *= f.nrows; f.nrows = 1; }   // the fill kernel counts a row in 32 bits
  f.dst_rank = q.dev; f.dst_phys = device_map[q.dev]; f.kind = kind;
  const unsigned long long slot = atomicAdd(reinterpret_cast<unsigned long long*>(&totals->n_fills), 1ull);
  fills[slot] = f;
  atomicAdd(reinterpret_cast<unsigned long long*>(&totals->fill_bytes), (unsigned long long)((int64_t)(r1 - r0) * q.nc * es));
}

// Bounds check of the finished plan (a safety net of our own: compute-sanitizer is not available everywhere): every
// chunk's source, destination and staging extent must lie inside the buffer it addresses.  One thread per chunk.
// staged: 1 / 0 for the plan's two lists, -1 for an address-ordered list (each record says which it is).  `sum` receives
// an order-independent checksum of the records, so that the ordered lists can be checked to be permutations of the
// plan's lists.
__device__ __forceinline__ unsigned long long mix64(unsigned long long x) {
  x ^= x >> 33; x *= 0xff51afd7ed558ccdull; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull; x ^= x >> 33; return x;
}
__global__ void __launch_bounds__(256)
plan_validate_kernel(const Chunk* __restrict__ ch, long long n, int staged_list, const int64_t* __restrict__ old_bytes,
                     const int64_t* __restrict__ new_bytes, int64_t staging_bytes, unsigned long long* __restrict__ bad,
                     unsigned long long* __restrict__ sum) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = i < n;                                       // every lane stays for the warp reduction below
  const Chunk c = ch[live ? i : 0];
  const bool staged = staged_list < 0 ? (c.pad & CHUNK_STAGED) != 0 : staged_list != 0;
  const int64_t span_src = (int64_t)(c.nrows - 1) * c.src_stride + c.row_bytes;
  const int64_t span_dst = (int64_t)(c.nrows - 1) * c.dst_stride + c.row_bytes;
  bool ok = c.nrows >= 1 && c.row_bytes >= 1 && (int64_t)c.nrows * c.row_bytes <= ETC_CHUNK_BYTES;
  ok = ok && c.src_off >= 0 && c.src_off + span_src <= old_bytes[c.src_buf];
  ok = ok && c.dst_off >= 0 && c.dst_off + span_dst <= new_bytes[c.dst_buf];
  ok = ok && (c.nrows == 1 || (c.src_stride >= c.row_bytes && c.dst_stride >= c.row_bytes));
  if (staged) ok = ok && c.stg_off >= 0 && c.stg_off + (int64_t)c.nrows * c.row_bytes <= staging_bytes;
  if (c.vec > 1) {
    int64_t al = c.src_off | c.dst_off | c.row_bytes | (staged ? c.stg_off : 0);
    if (c.nrows > 1) al |= (int64_t)c.src_stride | (int64_t)c.dst_stride;
    ok = ok && (al & (c.vec - 1)) == 0;
  }
  if (live && !ok) atomicAdd(bad, 1ull);
  unsigned long long h = mix64((unsigned long long)c.src_off ^ mix64((unsigned long long)c.dst_off ^ mix64((unsigned long long)c.stg_off)));
  h = mix64(h ^ ((unsigned long long)(uint32_t)c.src_stride << 32 | (uint32_t)c.dst_stride));
  h = mix64(h ^ ((unsigned long long)(uint32_t)c.row_bytes << 32 | (uint32_t)c.nrows));
  h = mix64(h ^ ((unsigned long long)c.src_buf << 32 | (unsigned long long)c.dst_buf << 16 | (unsigned long long)(uint16_t)c.vec) ^ (staged ? 0x9e3779b97f4a7c15ull : 0));
  if (!live) h = 0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) h += __shfl_xor_sync(0xffffffffu, h, o);
  if ((threadIdx.x & 31) == 0 && h) atomicAdd(sum, h);
}

}  // namespace etc

using namespace etc;

cudaError_t etc::plan_use(const etc_plan* pl, cudaStream_t st) {
  cudaError_t e = cudaSuccess;
  if (st != pl->stream_created_on && pl->ready) {
    // inside a stream capture the wait becomes an external-event node of the graph (a plain wait on an event recorded
    // outside the capture is not allowed there)
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    e = cudaStreamIsCapturing(st, &cap);
    if (e == cudaSuccess)
      e = cudaStreamWaitEvent(st, pl->ready, cap == cudaStreamCaptureStatusActive ? cudaEventWaitExternal : cudaEventWaitDefault);
  }
  pl->streams.note(st);
  return e;
}

// pinned slots for the totals read-back (a pageable destination would make the copy synchronous and slower)
static PlanTotals* g_pinned_totals = nullptr;
static unsigned g_pinned_next = 0;
constexpr unsigned N_PINNED_TOTALS = 64;

static bool on_device_ptr(const void* p) {
  cudaPointerAttributes attr{};
  if (cudaPointerGetAttributes(&attr, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
  return attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged;
}

const PlanTotals& etc::plan_totals(const etc_plan* cpl, etc_status* rc) {
  etc_plan* pl = const_cast<etc_plan*>(cpl);
  std::lock_guard<std::mutex> lock(pl->resolve_mu);
  if (!pl->resolved) {
    etc_status st = ETC_OK;
    cudaError_t e = pl->ready ? cudaEventSynchronize(pl->ready) : cudaStreamSynchronize(pl->stream_created_on);
    if (e == cudaSuccess) e = cudaMemcpy(&pl->totals, pl->d_totals, sizeof(PlanTotals), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { set_error_detail("plan totals read-back", e); st = ETC_ERR_CUDA; }
    else if (pl->totals.bad_map) st = ETC_ERR_BAD_MAP;
    else if (pl->totals.overflow) st = ETC_ERR_WORKSPACE;
    else if (pl->totals.local_bytes + pl->totals.remote_bytes + pl->totals.fill_bytes != pl->need_bytes) st = ETC_ERR_UNRECOVERABLE;
    pl->resolve_status = st;
    pl->resolved = true;
  }
  if (rc) *rc = pl->resolve_status;
  return pl->totals;
}

extern "C" etc_status etc_plan_create(const etc_layout* old_l, const etc_layout* new_l, const int32_t* device_map,
                                      int32_t flags, etc_plan** out, void* stream) {
  return etc_plan_create_failed(old_l, new_l, device_map, nullptr, flags, out, stream);
}

// Upper bounds of a plan's tables from what the host knows about the two layouts (ETC_NO_SYNC):
//   slices: a slice comes from one (new piece, old piece) pair of the same (kind, tensor) group — at most 4 of them when
//           the old kind is DP-sharded (the destination's own flat range is cut out of the rectangle), else 1;
//   chunks (per list): every slice ends in at most one short chunk, and every other chunk carries more than
//           ETC_CHUNK_BYTES / 2 bytes — or, on the re-aligning path, more than 4 KB (rows_per_chunk);
//   staging: payload + 16 bytes of padding per slice + 512 per (kind, source, destination) segment.
constexpr int64_t NO_SYNC_MAX_CHUNKS = 32768;
constexpr int64_t ORDER_MIN_LAZY_BYTES = 128ll << 20;      // about the size of the L2: below it DRAM locality is moot
static void plan_bounds(const etc_layout* old_l, const etc_layout* new_l, int K, etc_plan* pl) {
  const int nT = old_l->t.n_tensors;
  const bool old_sharded = old_l->cfg.dist_opt && old_l->cfg.dp > 1;
  int64_t sl = 0;
  for (size_t g = 0; g < old_l->grp_pieces.size() && g < new_l->grp_pieces.size(); ++g)
    sl += (int64_t)old_l->grp_pieces[g] * new_l->grp_pieces[g] * ((old_sharded && (int)(g / nT) >= 1) ? 4 : 1);
  const int64_t need = new_l->total_bytes;
  const int64_t min_pay = (old_l->aligned16 && new_l->aligned16) ? ETC_CHUNK_BYTES / 2 : 4096;
  pl->bound_slices = sl + 1;
  pl->bound_chunks = sl + need / min_pay + 2;
  pl->bound_staging = need + 16 * sl + 512ll * K * old_l->t.n_dev * new_l->t.n_dev + 512;
  pl->need_bytes = need;
}

extern "C" int64_t etc_staging_bound(const etc_layout* old_l, const etc_layout* new_l, int32_t flags) {
  if (!old_l || !new_l || !etc_same_model(old_l, new_l)) return ETC_ERR_INVALID_ARG;
  if (flags & ETC_ALL_DIRECT) return 0;
  etc_plan tmp;
  plan_bounds(old_l, new_l, (flags & ETC_KIND_MAJOR) ? ETC_NUM_KINDS : 1, &tmp);
  return tmp.bound_staging;
}

extern "C" etc_status etc_plan_create_failed(const etc_layout* old_l, const etc_layout* new_l, const int32_t* device_map,
                                             const uint8_t* failed, int32_t flags, etc_plan** out, void* stream) {
  clear_error_detail();
  if (!old_l || !new_l || !device_map || !out) return ETC_ERR_INVALID_ARG;
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (flags < 0 || flags > (ETC_ALL_STAGED | ETC_KIND_MAJOR | ETC_ALL_DIRECT | ETC_NO_SYNC | ETC_NO_REORDER)) return ETC_ERR_INVALID_ARG;
  if ((flags & ETC_ALL_STAGED) && (flags & ETC_ALL_DIRECT)) return ETC_ERR_INVALID_ARG;
  if (!etc_same_model(old_l, new_l)) return ETC_ERR_MISMATCH;
  const int n_old = old_l->t.n_dev, n_new = new_l->t.n_dev, P = n_old > n_new ? n_old : n_new;
  if ((long long)P * ETC_NUM_KINDS > 65535) return ETC_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  ETC_CUDA_TRY(layout_use(old_l, st));
  ETC_CUDA_TRY(layout_use(new_l, st));
  const int K = (flags & ETC_KIND_MAJOR) ? ETC_NUM_KINDS : 1;
  const long long U = (long long)K * n_old * n_new;
  // sub-blocks per unit: enough warps to fill the machine when there are few units, 1 when there are many
  const int want = (new_l->max_dev_pieces / K + 31) / 32;
  const int B = (int)std::max<long long>(1, std::min<long long>(want, 65536 / U));

  etc_plan* pl = new etc_plan();
  pl->n_old = n_old; pl->n_new = n_new; pl->P = P; pl->flags = flags & ~(ETC_NO_SYNC | ETC_NO_REORDER); pl->stream_created_on = st;
  pl->streams.note(st);
  pl->old_bytes.assign(old_l->h_buffer_bytes, old_l->h_buffer_bytes + (size_t)n_old * ETC_NUM_KINDS);
  pl->new_bytes.assign(new_l->h_buffer_bytes, new_l->h_buffer_bytes + (size_t)n_new * ETC_NUM_KINDS);
  plan_bounds(old_l, new_l, K, pl);
  // reading A31: the new layout's padded vocabulary has rows the old one lacks -> those are zero-filled
  const bool grows = new_l->vocab_rows > old_l->vocab_rows && new_l->n_emb_pieces > 0;
  pl->bound_fills = grows ? new_l->n_emb_pieces : 0;
  // ETC_NO_SYNC is honoured while the bound-sized grids stay small: every CTA of a copy launch beyond the real chunk
  // count costs ~0.7 us of an SM's three CTA slots (it reads the count and leaves), and the bound is about twice the
  // real count — measured on c2 (196 K bound, 91 K real) the surplus cost 0.17 ms per call where the one host sync of an
  // exact plan costs 0.02 ms.  Up to NO_SYNC_MAX_CHUNKS the surplus is worth less than a sync (states up to ~1 GB).
  const bool lazy = (flags & ETC_NO_SYNC) && pl->bound_chunks <= NO_SYNC_MAX_CHUNKS;
  pl->lazy = lazy; pl->resolved = !lazy;
  auto fail = [&](etc_status s) { etc_plan_destroy(pl); return s; };
#define PLAN_TRY(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) { set_error_detail(#expr, _e); return fail(ETC_ERR_CUDA); } } while (0)

  // device_map may live on the host or on the device
  const bool on_device = on_device_ptr(device_map);
  if (!on_device) {
    std::vector<char> seen((size_t)P, 0);
    for (int n = 0; n < n_new; ++n) {
      const int p = device_map[n];
      if (p < 0 || p >= P || seen[p]) return fail(ETC_ERR_BAD_MAP);
      seen[p] = 1;
    }
  }
  // workspace blob 1: bases | blocks | traffic | totals | map | pointer tables | failure mask | zero-fill list
  auto al = [](size_t x) { return (x + 255) & ~size_t(255); };
  const size_t o_bases = 0, o_blocks = o_bases + al(sizeof(UnitBase) * (size_t)U),
               o_traffic = o_blocks + al(sizeof(BlockCount) * (size_t)U * B),
               o_totals = o_traffic + al(sizeof(int64_t) * (size_t)P * P), o_map = o_totals + al(sizeof(PlanTotals)),
               o_ptrs = o_map + al(sizeof(int32_t) * (size_t)n_new),
               o_failed = o_ptrs + al(sizeof(void*) * (size_t)(n_old + n_new) * ETC_NUM_KINDS),
               o_fills = o_failed + al((size_t)n_old),
               ws_bytes = o_fills + (grows ? al(sizeof(etc_slice) * (size_t)new_l->n_emb_pieces) : 0);
  PLAN_TRY(cudaMallocAsync(&pl->d_ws, ws_bytes, st));
  char* ws = static_cast<char*>(pl->d_ws);
  pl->d_bases = reinterpret_cast<UnitBase*>(ws + o_bases);
  pl->d_blocks = reinterpret_cast<BlockCount*>(ws + o_blocks); pl->d_traffic = reinterpret_cast<int64_t*>(ws + o_traffic);
  pl->d_totals = reinterpret_cast<PlanTotals*>(ws + o_totals); pl->d_map = reinterpret_cast<int32_t*>(ws + o_map);
  pl->d_ptrs = reinterpret_cast<void**>(ws + o_ptrs);
  // metadata moves as kernels on `st`, never through the copy engines (xfer.cu).  A device map is read in place by the
  // count and scan kernels; the scan kernel keeps a copy in the plan, which everything later uses.
  const int32_t* map_in = device_map;
  if (!on_device) { PLAN_TRY(write_small(pl->d_map, device_map, sizeof(int32_t) * (size_t)n_new, st)); map_in = pl->d_map; }
  const uint8_t* d_failed = nullptr;
  if (failed) {                                                 // reading A26: host or device mask [n_old]
    if (on_device_ptr(failed)) PLAN_TRY(copy_by_kernel(ws + o_failed, failed, (size_t)n_old, st));
    else PLAN_TRY(write_small(ws + o_failed, failed, (size_t)n_old, st));
    d_failed = reinterpret_cast<const uint8_t*>(ws + o_failed);
  }

  const unsigned grid = (unsigned)((U * B + PLAN_WARPS - 1) / PLAN_WARPS);
  plan_count_kernel<<<grid, PLAN_WARPS * 32, 0, st>>>(old_l->t, new_l->t, map_in, d_failed, K, B, pl->d_blocks);
  PLAN_TRY(cudaGetLastError());
  PlanTotals* h_tot = nullptr;                                  // pinned slot for the totals read-back (not for no-sync plans)
  if (!lazy) {
    {
      static std::mutex mu;                                     // plans may be created from several host threads
      std::lock_guard<std::mutex> lock(mu);
      if (!g_pinned_totals) PLAN_TRY(cudaMallocHost(&g_pinned_totals, sizeof(PlanTotals) * N_PINNED_TOTALS));
    }
    h_tot = &g_pinned_totals[__atomic_fetch_add(&g_pinned_next, 1u, __ATOMIC_RELAXED) % N_PINNED_TOTALS];
  }
  plan_scan_kernel<<<1, SCAN_THREADS, 0, st>>>(pl->d_blocks, B, U, K, n_old, n_new, P, pl->flags, map_in, pl->d_map,
                                               pl->d_bases, pl->d_traffic, pl->d_totals, grows ? nullptr : h_tot,
                                               lazy ? pl->bound_slices : 0, pl->bound_chunks, pl->bound_staging);
  PLAN_TRY(cudaGetLastError());
  count_launch(2);
  if (grows) {
    pl->d_fills = reinterpret_cast<etc_slice*>(ws + o_fills);
    plan_fills_kernel<<<(unsigned)((new_l->t.n_pieces + 255) / 256), 256, 0, st>>>(new_l->t, pl->d_map, old_l->vocab_rows,
                                                                                   new_l->lm_head_id, pl->d_fills, pl->d_totals);
    PLAN_TRY(cudaGetLastError());
    count_launch();
  }
  int64_t n_sl_s, n_sl_l, n_ch_s, n_ch_l;                       // table capacities
  if (!lazy) {
    // the scan kernel wrote the totals straight into the pinned slot, unless the zero-fill kernel still had to add to them
    if (grows) PLAN_TRY(copy_by_kernel(h_tot, pl->d_totals, sizeof(PlanTotals), st));
    PLAN_TRY(cudaStreamSynchronize(st));                        // the one host sync: sizes must come back
    pl->totals = *h_tot;
    if (pl->totals.bad_map) return fail(ETC_ERR_BAD_MAP);
    // every needed byte must have found its one source
    if (pl->totals.local_bytes + pl->totals.remote_bytes + pl->totals.fill_bytes != pl->need_bytes) return fail(ETC_ERR_UNRECOVERABLE);
    n_sl_s = pl->totals.n_slices_staged; n_sl_l = pl->totals.n_slices_local;
    n_ch_s = pl->totals.n_chunks_staged; n_ch_l = pl->totals.n_chunks_local;
  } else {
    n_sl_s = n_sl_l = pl->bound_slices; n_ch_s = n_ch_l = pl->bound_chunks;
  }

  // blob 2: slice records | chunk descriptors
  const size_t o_sls = 0, o_sll = o_sls + al(sizeof(etc_slice) * (size_t)n_sl_s),
               o_chs = o_sll + al(sizeof(etc_slice) * (size_t)n_sl_l), o_chl = o_chs + al(sizeof(Chunk) * (size_t)n_ch_s),
               tb_bytes = o_chl + al(sizeof(Chunk) * (size_t)n_ch_l);
  if (tb_bytes) {
    PLAN_TRY(cudaMallocAsync(&pl->d_tb, tb_bytes, st));
    char* tb = static_cast<char*>(pl->d_tb);
    pl->d_sl_staged = reinterpret_cast<etc_slice*>(tb + o_sls); pl->d_sl_local = reinterpret_cast<etc_slice*>(tb + o_sll);
    pl->d_ch_staged = reinterpret_cast<Chunk*>(tb + o_chs); pl->d_ch_local = reinterpret_cast<Chunk*>(tb + o_chl);
  }
  if (n_sl_s + n_sl_l) {
    plan_fill_kernel<<<grid, PLAN_WARPS * 32, 0, st>>>(old_l->t, new_l->t, pl->d_map, d_failed, pl->flags, K, B, pl->d_blocks,
                                                       pl->d_bases, pl->d_sl_staged, pl->d_sl_local, pl->d_ch_staged,
                                                       pl->d_ch_local, lazy ? pl->d_totals : nullptr);
    PLAN_TRY(cudaGetLastError());
    count_launch();
  }
  // the launch lists in address order (plan_order.cu).  A bound-sized ETC_NO_SYNC plan gets them only if it moves enough
  // for the order to matter (a state that fits the L2 gains nothing; its four extra launches would be a tenth of
  // the whole migration)
  if (!(flags & ETC_NO_REORDER) && (!lazy || pl->need_bytes >= ORDER_MIN_LAZY_BYTES))
    PLAN_TRY(plan_build_order(pl, n_ch_s, n_ch_l, st, lazy ? pl->d_totals : nullptr));
  // the tables are complete once `st` reaches this point: readers on other streams wait for it (plan_use)
  PLAN_TRY(cudaEventCreateWithFlags(&pl->ready, cudaEventDisableTiming));
  PLAN_TRY(cudaEventRecord(pl->ready, st));
#undef PLAN_TRY
  *out = pl;
  return ETC_OK;
}

extern "C" void etc_plan_destroy(etc_plan* pl) {
  if (!pl) return;
  etc::DeviceGuard device_guard;
  cudaStream_t st = pl->streams.join(pl->stream_created_on);
  if (pl->d_ws) cudaFreeAsync(pl->d_ws, st);
  if (pl->d_tb) cudaFreeAsync(pl->d_tb, st);
  if (pl->d_rounds_ws) cudaFreeAsync(pl->d_rounds_ws, st);
  if (pl->d_order_ws) cudaFreeAsync(pl->d_order_ws, st);
  if (pl->d_round_order_ws) cudaFreeAsync(pl->d_round_order_ws, st);
  if (pl->ready) cudaEventDestroy(pl->ready);
  delete pl;
}

extern "C" int32_t etc_plan_is_deferred(const etc_plan* pl) {
  if (!pl) return ETC_ERR_INVALID_ARG;
  return pl->lazy ? 1 : 0;
}

extern "C" etc_status etc_plan_get_stats(const etc_plan* pl, etc_plan_stats* out) {
  if (!pl || !out) return ETC_ERR_INVALID_ARG;
  etc_status rc = ETC_OK;
  const PlanTotals& t = plan_totals(pl, &rc);                   // an ETC_NO_SYNC plan is waited for here
  if (rc != ETC_OK) return rc;
  out->staging_bytes = t.staging_bytes; out->local_bytes = t.local_bytes; out->remote_bytes = t.remote_bytes;
  out->staged_bytes = (pl->flags & ETC_ALL_STAGED) ? t.local_bytes + t.remote_bytes : ((pl->flags & ETC_ALL_DIRECT) ? 0 : t.remote_bytes);
  out->n_slices_local = t.n_slices_local; out->n_slices_staged = t.n_slices_staged;
  out->n_chunks_local = t.n_chunks_local; out->n_chunks_staged = t.n_chunks_staged;
  out->n_old = pl->n_old; out->n_new = pl->n_new; out->P = pl->P; out->flags = pl->flags;
  out->fill_bytes = t.fill_bytes; out->n_fills = t.n_fills;
  return ETC_OK;
}

extern "C" etc_status etc_plan_get_traffic(const etc_plan* pl, int64_t* h_traffic) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !h_traffic) return ETC_ERR_INVALID_ARG;
  { etc_status rc = ETC_OK; plan_totals(pl, &rc); if (rc != ETC_OK) return rc; }   // a device-detected error of an ETC_NO_SYNC plan
  ETC_CUDA_TRY(cudaStreamSynchronize(pl->stream_created_on));
  ETC_CUDA_TRY(cudaMemcpy(h_traffic, pl->d_traffic, sizeof(int64_t) * (size_t)pl->P * pl->P, cudaMemcpyDeviceToHost));
  return ETC_OK;
}

extern "C" etc_status etc_plan_get_map(const etc_plan* pl, int32_t* h_device_map) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !h_device_map) return ETC_ERR_INVALID_ARG;
  ETC_CUDA_TRY(cudaStreamSynchronize(pl->stream_created_on));
  ETC_CUDA_TRY(cudaMemcpy(h_device_map, pl->d_map, sizeof(int32_t) * (size_t)pl->n_new, cudaMemcpyDeviceToHost));
  return ETC_OK;
}

extern "C" etc_status etc_plan_get_slices(const etc_plan* pl, int32_t which, etc_slice* h_out) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !h_out || (which != 0 && which != 1)) return ETC_ERR_INVALID_ARG;
  etc_status rc = ETC_OK;
  const PlanTotals& t = plan_totals(pl, &rc);
  if (rc != ETC_OK) return rc;
  const int64_t n = which == 0 ? t.n_slices_staged : t.n_slices_local;
  const etc_slice* src = which == 0 ? pl->d_sl_staged : pl->d_sl_local;
  ETC_CUDA_TRY(cudaStreamSynchronize(pl->stream_created_on));
  if (n) ETC_CUDA_TRY(cudaMemcpy(h_out, src, sizeof(etc_slice) * (size_t)n, cudaMemcpyDeviceToHost));
  return ETC_OK;
}

static_assert(sizeof(etc_chunk) == sizeof(etc::Chunk), "etc_chunk mirrors Chunk");
extern "C" etc_status etc_plan_get_chunks(const etc_plan* pl, int32_t which, etc_chunk* h_out) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !h_out || which < 0 || which > 3) return ETC_ERR_INVALID_ARG;
  etc_status rc = ETC_OK;
  const PlanTotals& t = plan_totals(pl, &rc);
  if (rc != ETC_OK) return rc;
  const Chunk* src = which == 0 ? pl->d_ch_staged : which == 1 ? pl->d_ch_local : which == 2 ? pl->d_ch1 : pl->d_ch2;
  const int64_t n = which == 1 ? t.n_chunks_local : which == 2 ? t.n_chunks_staged + t.n_chunks_local : t.n_chunks_staged;
  if (which >= 2 && !pl->d_ch1) return ETC_ERR_INVALID_ARG;
  ETC_CUDA_TRY(cudaStreamSynchronize(pl->stream_created_on));
  if (n) ETC_CUDA_TRY(cudaMemcpy(h_out, src, sizeof(Chunk) * (size_t)n, cudaMemcpyDeviceToHost));
  return ETC_OK;
}

extern "C" etc_status etc_plan_get_fills(const etc_plan* pl, etc_slice* h_out) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !h_out) return ETC_ERR_INVALID_ARG;
  etc_status rc = ETC_OK;
  const int64_t nf = plan_totals(pl, &rc).n_fills;
  if (rc != ETC_OK) return rc;
  ETC_CUDA_TRY(cudaStreamSynchronize(pl->stream_created_on));
  if (nf) ETC_CUDA_TRY(cudaMemcpy(h_out, pl->d_fills, sizeof(etc_slice) * (size_t)nf, cudaMemcpyDeviceToHost));
  return ETC_OK;
}

extern "C" etc_status etc_plan_validate(const etc_plan* pl, int64_t* n_bad, void* stream) {
  clear_error_detail();
  etc::DeviceGuard device_guard;                 // the library's device for this call; the caller's is restored on return
  if (device_guard.err != cudaSuccess) { etc::set_error_detail("cudaSetDevice", device_guard.err); return ETC_ERR_CUDA; }
  if (!pl || !n_bad) return ETC_ERR_INVALID_ARG;
  etc_status plan_rc = ETC_OK;
  const PlanTotals& t = plan_totals(pl, &plan_rc);
  if (plan_rc != ETC_OK) return plan_rc;                        // an unusable ETC_NO_SYNC plan has nothing to validate
  cudaStream_t st = (cudaStream_t)stream;
  ETC_CUDA_TRY(plan_use(pl, st));
  const size_t ns = pl->old_bytes.size(), nd = pl->new_bytes.size();
  int64_t* d_sizes = nullptr;
  ETC_CUDA_TRY(cudaMallocAsync(&d_sizes, sizeof(int64_t) * (ns + nd + 7), st));
  auto done = [&](etc_status rc) { cudaFreeAsync(d_sizes, st); return rc; };
#define VAL_TRY(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) { set_error_detail(#expr, _e); return done(ETC_ERR_CUDA); } } while (0)
  VAL_TRY(cudaMemcpyAsync(d_sizes, pl->old_bytes.data(), sizeof(int64_t) * ns, cudaMemcpyHostToDevice, st));
  VAL_TRY(cudaMemcpyAsync(d_sizes + ns, pl->new_bytes.data(), sizeof(int64_t) * nd, cudaMemcpyHostToDevice, st));
  // d_bad[0] = bad chunks; [1], [2] checksums of the staged / local list; [3], [4] of the ordered launch lists; [5], [6]
  // of the per-round ordered lists
  unsigned long long* d_bad = reinterpret_cast<unsigned long long*>(d_sizes + ns + nd);
  VAL_TRY(cudaMemsetAsync(d_bad, 0, 7 * sizeof(unsigned long long), st));
  auto check = [&](const Chunk* list, long long n, int staged, int slot) -> cudaError_t {
    if (!n || !list) return cudaSuccess;
    plan_validate_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(list, n, staged, d_sizes, d_sizes + ns, t.staging_bytes, d_bad,
                                                                       d_bad + slot);
    count_launch();
    return cudaGetLastError();
  };
  VAL_TRY(check(pl->d_ch_staged, t.n_chunks_staged, 1, 1));
  VAL_TRY(check(pl->d_ch_local, t.n_chunks_local, 0, 2));
  VAL_TRY(check(pl->d_ch1, t.n_chunks_staged + t.n_chunks_local, -1, 3));
  VAL_TRY(check(pl->d_ch2, t.n_chunks_staged, 1, 4));
  VAL_TRY(check(pl->d_rch1, t.n_chunks_staged + t.n_chunks_local, -1, 5));
  VAL_TRY(check(pl->d_rch2, t.n_chunks_staged, 1, 6));
  unsigned long long h[7] = {0, 0, 0, 0, 0, 0, 0};
  VAL_TRY(cudaMemcpyAsync(h, d_bad, sizeof(h), cudaMemcpyDeviceToHost, st));
  VAL_TRY(cudaStreamSynchronize(st));
  // the ordered lists must hold exactly the plan's chunks (order-independent checksums)
  if (pl->d_ch1 && h[3] != h[1] + h[2]) h[0] += 1;
  if (pl->d_ch2 && t.n_chunks_staged && h[4] != h[1]) h[0] += 1;
  if (pl->d_rch1 && h[5] != h[1] + h[2]) h[0] += 1;
  if (pl->d_rch2 && t.n_chunks_staged && h[6] != h[1]) h[0] += 1;
  const unsigned long long h_bad = h[0];
#undef VAL_TRY
  *n_bad = (int64_t)h_bad;
  return done(ETC_OK);
}
