"""ctypes wrapper around oracle/etc_oracle.c — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this.
It never imports paper_2607_04749_b200 (the CUDA path) and shares no code with it.

`build()` compiles etc_oracle.c with gcc (OpenMP) into oracle/liboracle.so.
"""
from __future__ import annotations
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "etc_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


class Model(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("style", "n_layers", "hidden", "n_q_heads", "n_kv_heads", "head_dim",
                                          "ffn_hidden", "vocab", "max_pos", "tied", "param_bytes", "kinds", "qkv_order")]


class Cfg(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("tp", "pp", "dp", "dist_opt", "pp_first", "pp_last", "dist_opt_align",
                                          "vocab_divisor")]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        P = C.POINTER
        L.orc_num_logical.restype = i32
        L.orc_logical_info.restype = i32
        L.orc_kind_bytes.restype = i32
        L.orc_layout_new.restype = i32
        L.orc_layout_new.argtypes = [P(Model), P(Cfg), P(vp)]
        L.orc_layout_free.argtypes = [vp]
        L.orc_layout_free.restype = None
        L.orc_layout_set_failed.argtypes = [vp, vp]
        L.orc_layout_set_failed.restype = None
        L.orc_num_devices.restype = i32
        L.orc_num_devices.argtypes = [vp]
        L.orc_buffer_elems.restype = i64
        L.orc_buffer_elems.argtypes = [vp, i32, i32]
        L.orc_global_of_range.restype = i32
        L.orc_global_of_range.argtypes = [vp, i32, i32, i64, i64, vp, vp, vp, vp]
        L.orc_holders_of.restype = i32
        L.orc_holders_of.argtypes = [vp, i32, i32, i64, i64, i32, vp, vp]
        L.orc_overlap_elementwise.restype = i32
        L.orc_overlap_elementwise.argtypes = [vp, vp, i32, vp, vp, vp]
        L.orc_overlap_ranges.restype = i32
        L.orc_overlap_ranges.argtypes = [vp, vp, vp, vp, vp]
        L.orc_sketch_bruteforce.restype = i64
        L.orc_sketch_bruteforce.argtypes = [vp, i32, i32, vp, vp, P(i64)]
        L.orc_sketch_hungarian.restype = i32
        L.orc_sketch_hungarian.argtypes = [vp, i32, i32, vp, vp, P(i64)]
        L.orc_source_of.restype = i32
        L.orc_source_of.argtypes = [vp, vp, vp, i32, i32, vp, i64, vp, vp]
        L.orc_migrate_range.restype = i32
        L.orc_migrate_range.argtypes = [vp, vp, vp, i32, i32, i64, i64, vp, vp, vp, vp, vp]
        L.orc_migrate.restype = i32
        L.orc_migrate.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.orc_migrate_fill.restype = i32
        L.orc_migrate_fill.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
        L.orc_logical_info_cfg.restype = i32
        L.orc_logical_info_cfg.argtypes = [P(Model), P(Cfg), vp, vp, vp, vp, vp]
        L.orc_max_threads.restype = i32
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"oracle error {code}")
        self.code = code


def _model(m: dict) -> Model:
    return Model(**{k: int(m.get(k, 0)) for k, _ in Model._fields_})


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def max_threads() -> int:
    return int(lib().orc_max_threads())


def _cfg(cfg: dict) -> Cfg:
    return Cfg(**{k: int(cfg.get(k, 0)) for k, _ in Cfg._fields_})


def logical_tensors(model: dict, cfg: dict | None = None):
    """[(rows, cols, split, where, layer)] for every logical tensor, in id order.  With cfg: the embedding tensors have
    that parallel configuration's padded vocabulary rows (reading A31); without: the unpadded model."""
    m = _model(model)
    n = lib().orc_num_logical(C.byref(m))
    rows = np.zeros(n, np.int64); cols = np.zeros(n, np.int64)
    split = np.zeros(n, np.int32); where = np.zeros(n, np.int32); layer = np.zeros(n, np.int32)
    c = _cfg(cfg) if cfg is not None else None
    lib().orc_logical_info_cfg(C.byref(m), C.byref(c) if c is not None else None, _ptr(rows), _ptr(cols), _ptr(split),
                               _ptr(where), _ptr(layer))
    return [(int(rows[i]), int(cols[i]), int(split[i]), int(where[i]), int(layer[i])) for i in range(n)]


def kind_bytes(model: dict, kind: int) -> int:
    m = _model(model)
    return int(lib().orc_kind_bytes(C.byref(m), kind))


class Layout:
    """Oracle-side layout of one (model, parallel config)."""

    def __init__(self, model: dict, cfg: dict):
        self.model, self.cfg = dict(model), dict(cfg)
        m = _model(model)
        c = _cfg(cfg)
        h = C.c_void_p()
        rc = lib().orc_layout_new(C.byref(m), C.byref(c), C.byref(h))
        if rc:
            raise OracleError(rc)
        self.h = h
        self.n_dev = int(lib().orc_num_devices(h))

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_layout_free(self.h)
            self.h = None

    def set_failed(self, failed):
        """Mark devices of this (old) layout as failed (reading A26); None clears the mask."""
        if failed is None:
            lib().orc_layout_set_failed(self.h, None)
            self.failed = None
        else:
            f = np.ascontiguousarray(failed, np.uint8)
            assert f.shape == (self.n_dev,)
            lib().orc_layout_set_failed(self.h, _ptr(f))
            self.failed = f.copy()

    def kinds(self):
        return [k for k in range(4) if (self.model["kinds"] >> k) & 1]

    def logical_tensors(self):
        """the logical tensor list as this layout sees it (padded vocabulary rows, reading A31)"""
        return logical_tensors(self.model, self.cfg)

    def elem_bytes(self, kind):
        return kind_bytes(self.model, kind)

    def buffer_elems(self, dev, kind) -> int:
        return int(lib().orc_buffer_elems(self.h, dev, kind))

    def global_of(self, dev, kind, l0=0, count=None):
        """(lt, post_copy, row, col) arrays for local indices [l0, l0+count)."""
        if count is None:
            count = self.buffer_elems(dev, kind) - l0
        lt = np.zeros(count, np.int32); pc = np.zeros(count, np.int32)
        row = np.zeros(count, np.int64); col = np.zeros(count, np.int64)
        rc = lib().orc_global_of_range(self.h, dev, kind, l0, count, _ptr(lt), _ptr(pc), _ptr(row), _ptr(col))
        if rc:
            raise OracleError(rc)
        return lt, pc, row, col

    def holders_of(self, kind, lt, row, col):
        cap = 2 * self.n_dev + 2
        dev = np.zeros(cap, np.int32); l = np.zeros(cap, np.int64)
        n = lib().orc_holders_of(self.h, kind, lt, row, col, cap, _ptr(dev), _ptr(l))
        return [(int(dev[i]), int(l[i])) for i in range(n)]

    # ---- data helpers built on global_of + plain numpy indexing
    def shard_from_logical(self, dev, kind, logical: list) -> np.ndarray:
        """Buffer (dev, kind) cut out of the logical tensors (list of 2-D arrays indexed by tensor id)."""
        lt, _, row, col = self.global_of(dev, kind)
        dt = np.uint16 if self.elem_bytes(kind) == 2 else np.uint32
        out = np.zeros(lt.shape[0], dt)
        # the buffer is a concatenation of tensor shards: one gather per run of equal tensor id
        cuts = np.concatenate(([0], np.flatnonzero(np.diff(lt)) + 1, [lt.shape[0]])) if lt.shape[0] else np.zeros(1, np.int64)
        for a, b in zip(cuts[:-1], cuts[1:]):
            out[a:b] = logical[int(lt[a])][row[a:b], col[a:b]]
        return out


def P_of(old: Layout, new: Layout) -> int:
    return max(old.n_dev, new.n_dev)


def overlap(old: Layout, new: Layout, only_layers: bool = False, method: str = "elementwise"):
    """(overlap[n_new][P], need[n_new], hold[P]) in bytes."""
    P = P_of(old, new)
    ov = np.zeros((new.n_dev, P), np.int64); need = np.zeros(new.n_dev, np.int64); hold = np.zeros(P, np.int64)
    if method == "elementwise":
        rc = lib().orc_overlap_elementwise(old.h, new.h, int(only_layers), _ptr(ov), _ptr(need), _ptr(hold))
    else:
        assert not only_layers
        rc = lib().orc_overlap_ranges(old.h, new.h, _ptr(ov), _ptr(need), _ptr(hold))
    if rc:
        raise OracleError(rc)
    return ov, need, hold


def mask_cross_dp(old: Layout, new: Layout, ov: np.ndarray) -> np.ndarray:
    """The paper's DP isolation (reading A5): a copy of `ov` with every cross-DP cell zeroed."""
    out = np.ascontiguousarray(ov, np.int64).copy()
    lib().orc_mask_cross_dp.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib().orc_mask_cross_dp.restype = C.c_int32
    rc = lib().orc_mask_cross_dp(old.h, new.h, _ptr(out))
    if rc:
        raise OracleError(rc)
    return out


def sketch_bruteforce(ov: np.ndarray, avail=None):
    ov = np.ascontiguousarray(ov, np.int64)
    n, P = ov.shape
    m = np.zeros(n, np.int32); val = C.c_int64()
    av = None if avail is None else np.ascontiguousarray(avail, np.uint8)
    cnt = lib().orc_sketch_bruteforce(_ptr(ov), n, P, _ptr(av), _ptr(m), C.byref(val))
    return m, int(val.value), int(cnt)


def sketch_hungarian(ov: np.ndarray, avail=None):
    ov = np.ascontiguousarray(ov, np.int64)
    n, P = ov.shape
    m = np.zeros(n, np.int32); val = C.c_int64()
    av = None if avail is None else np.ascontiguousarray(avail, np.uint8)
    rc = lib().orc_sketch_hungarian(_ptr(ov), n, P, _ptr(av), _ptr(m), C.byref(val))
    if rc:
        raise OracleError(rc)
    return m, int(val.value)


def source_of(old: Layout, new: Layout, device_map, n, kind, l_list):
    dm = np.ascontiguousarray(device_map, np.int32)
    ll = np.ascontiguousarray(l_list, np.int64)
    sd = np.zeros(ll.shape[0], np.int32); sl = np.zeros(ll.shape[0], np.int64)
    rc = lib().orc_source_of(old.h, new.h, _ptr(dm), n, kind, _ptr(ll), ll.shape[0], _ptr(sd), _ptr(sl))
    if rc:
        raise OracleError(rc)
    return sd, sl


def _ptr_table(bufs, n_dev):
    tab = (C.c_void_p * (n_dev * 4))()
    for (dev, kind), a in bufs.items():
        tab[dev * 4 + kind] = a.ctypes.data
    return tab


def migrate(old: Layout, new: Layout, device_map, src_bufs: dict | None, want_overrides=False, fill_out=None):
    """Element-wise migration.  src_bufs: {(old_dev, kind): 1-D uint16/uint32 array} or None (traffic only).
    Returns (dst_bufs {(n, kind): array} or None, T[P][P], overrides).  fill_out: optional int64 array [n_new] that
    receives the bytes of each new rank that have no source and are zero-filled (reading A31).  The destination buffers
    start out poisoned, so a zero in them was written.

    Orchestration only: small problems are one call of orc_migrate_fill (OpenMP over new ranks); larger ones hand
    element ranges of the new buffers to host threads, each range through orc_migrate_range_fill with its own traffic
    matrix, summed afterwards — the per-element code is the same."""
    P = P_of(old, new)
    dm = np.ascontiguousarray(device_map, np.int32)
    T = np.zeros((P, P), np.int64); ovr = C.c_int64(0)
    dst = None; st = None; dt = None
    if src_bufs is not None:
        st = _ptr_table(src_bufs, old.n_dev)
        dst = {}
        for n in range(new.n_dev):
            for k in new.kinds():
                cnt = new.buffer_elems(n, k)
                dst[(n, k)] = np.full(cnt, 0xA5A5, np.uint16) if new.elem_bytes(k) == 2 else np.full(cnt, 0xA5A5A5A5, np.uint32)
        dt = _ptr_table(dst, new.n_dev)
    if fill_out is not None:
        assert fill_out.dtype == np.int64 and fill_out.shape == (new.n_dev,) and fill_out.flags.c_contiguous
    total = sum(new.buffer_elems(n, k) for n in range(new.n_dev) for k in new.kinds())
    if total < _PARALLEL_MIN_ELEMS:
        rc = lib().orc_migrate_fill(old.h, new.h, _ptr(dm), st, dt, _ptr(T), C.byref(ovr) if want_overrides else None,
                                    _ptr(fill_out))
        if rc:
            raise OracleError(rc)
        return dst, T, int(ovr.value)
    # ---- large problem: element ranges over a thread pool (the C code runs outside the GIL)
    from concurrent.futures import ThreadPoolExecutor
    if orc_check_map(dm, new.n_dev, P):
        raise OracleError(-1)
    L = lib()
    L.orc_migrate_range_fill.restype = C.c_int32
    L.orc_migrate_range_fill.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int64,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    tasks = [(n, k, l0, min(new.buffer_elems(n, k), l0 + _PARALLEL_CHUNK))
             for n in range(new.n_dev) for k in new.kinds() for l0 in range(0, new.buffer_elems(n, k), _PARALLEL_CHUNK)]

    def one(t):
        n, k, l0, l1 = t
        Tt = np.zeros((P, P), np.int64); o = C.c_int64(0); f = C.c_int64(0)
        rc = L.orc_migrate_range_fill(old.h, new.h, _ptr(dm), n, k, l0, l1, st, _ptr(dst[(n, k)]) if dst is not None else None,
                                      _ptr(Tt), C.byref(o) if want_overrides else None, None, C.byref(f))
        return rc, Tt, int(o.value), n, int(f.value)

    if fill_out is not None:
        fill_out[:] = 0
    with ThreadPoolExecutor(os.cpu_count() or 1) as ex:
        for rc, Tt, o, n, f in ex.map(one, tasks):
            if rc:
                raise OracleError(rc)
            T += Tt
            ovr.value += o
            if fill_out is not None:
                fill_out[n] += f
    return dst, T, int(ovr.value)


_PARALLEL_MIN_ELEMS = 4_000_000
_PARALLEL_CHUNK = 1 << 19


def orc_check_map(dm, n_new, P) -> bool:
    """True if dm is not an injective map [0, n_new) -> [0, P) (what orc_migrate_fill rejects up front)."""
    return bool(((dm < 0) | (dm >= P)).any() or len(set(dm.tolist())) != n_new)


def migrate_range(old: Layout, new: Layout, device_map, n, kind, l0, l1, src_bufs: dict | None, dst=None,
                  T=None, written=None, src_windows: dict | None = None, dst_first: int = 0):
    """Element-wise migration of local indices [l0, l1) of new buffer (n, kind) (orc_migrate_range).  src_bufs:
    {(old_dev, kind): whole old buffer}.  src_windows (instead of src_bufs): {(old_dev, kind): (first, array)} where
    `array` holds only the elements [first, first + len(array)) of that old buffer — for callers that know which part of
    the old state a range reads and cannot hold all of it in host memory; the table entry is the address the whole
    buffer would start at, so elements outside the window must not be read.  dst_first: `dst` holds only the elements
    [dst_first, dst_first + len(dst)) of the new buffer (same address trick on the destination side; [l0, l1) must lie
    inside it) — orchestration only, the per-element C routine is the same."""
    dm = np.ascontiguousarray(device_map, np.int32)
    dst_p = _ptr(dst)
    if dst_first:
        assert dst is not None and dst_first <= l0 and l1 <= dst_first + dst.shape[0]
        dst_p = C.c_void_p(dst.ctypes.data - int(dst_first) * dst.itemsize)
    st = _ptr_table(src_bufs, old.n_dev) if src_bufs is not None else None
    if src_windows is not None:
        assert src_bufs is None
        st = (C.c_void_p * (old.n_dev * 4))()
        for (dev, k), (first, a) in src_windows.items():
            st[dev * 4 + k] = a.ctypes.data - int(first) * a.itemsize
    rc = lib().orc_migrate_range(old.h, new.h, _ptr(dm), n, kind, l0, l1, st, dst_p, _ptr(T), None, _ptr(written))
    if rc:
        raise OracleError(rc)
