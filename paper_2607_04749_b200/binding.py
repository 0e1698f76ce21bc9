"""ctypes binding of libetc.so (include/etc.h).  Same names as the C ABI; argument marshalling only.

torch is used for device memory and streams, nothing else: every step of the path runs in the library's kernels.
"""
from __future__ import annotations
import ctypes as C
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libetc.so")
_lib = None
_inited = False

ETC_LOCAL_DIRECT, ETC_ALL_STAGED, ETC_KIND_MAJOR, ETC_ALL_DIRECT, ETC_NO_SYNC, ETC_NO_REORDER = 0, 1, 2, 4, 8, 16
ETC_SKETCH_AUTO, ETC_SKETCH_EXHAUSTIVE, ETC_SKETCH_HUNGARIAN = 0, 1, 2
ETC_SKETCH_STATIC_MAX_P, ETC_SKETCH_STATIC_SCRATCH_BYTES = 1024, 28672
ETC_PHASE_PACK, ETC_PHASE_UNPACK, ETC_PHASE_ALL = 1, 2, 3
ETC_DEFRAG_OCCUPANCY, ETC_DEFRAG_EFFICIENCY, ETC_DEFRAG_BOTH = 1, 2, 3

EXPORTED_SYMBOLS = (
    "etc_init", "etc_layout_create", "etc_layout_destroy", "etc_layout_num_devices", "etc_layout_num_pieces",
    "etc_layout_buffer_bytes", "etc_cost_matrix", "etc_sketch", "etc_plan_create", "etc_plan_destroy",
    "etc_plan_get_stats", "etc_plan_get_traffic", "etc_plan_get_slices", "etc_plan_get_fills", "etc_migrate",
    "etc_migrate_phase",
    "etc_status_string", "etc_last_error_detail", "etc_kernel_launches", "etc_defrag",
    "etc_plan_set_rounds", "etc_plan_get_round", "etc_migrate_round", "etc_plan_create_failed", "etc_mask_failed",
    "etc_upload_sources", "etc_plan_validate", "etc_mask_cross_dp", "etc_staging_bound", "etc_migrate_state", "etc_plan_get_map",
    "etc_plan_get_chunks", "etc_sketch_static", "etc_plan_is_deferred",
)


class EtcError(RuntimeError):
    def __init__(self, code, detail=""):
        name = lib().etc_status_string(code).decode() if _lib is not None else str(code)
        super().__init__(f"{name} ({code}){': ' + detail if detail else ''}")
        self.code = code


class _ModelDesc(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("style", "n_layers", "hidden", "n_q_heads", "n_kv_heads", "head_dim",
                                          "ffn_hidden", "vocab", "max_pos", "tied_embeddings", "param_dtype", "kinds",
                                          "qkv_order")]


class _ParallelCfg(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("tp", "pp", "dp", "dist_opt", "pp_first", "pp_last", "dist_opt_align",
                                          "vocab_divisor")]


class _PlanStats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("staging_bytes", "local_bytes", "remote_bytes", "staged_bytes",
                                          "n_slices_local", "n_slices_staged", "n_chunks_local", "n_chunks_staged")] + \
               [(n, C.c_int32) for n in ("n_old", "n_new", "P", "flags")] + \
               [(n, C.c_int64) for n in ("fill_bytes", "n_fills")]


class _RoundInfo(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("kind", "sub", "n_sub", "pad")] + \
               [(n, C.c_int64) for n in ("staging_bytes", "staged_bytes", "local_bytes", "n_chunks_staged",
                                          "n_chunks_local")]


class _Slice(C.Structure):
    _fields_ = [("src_off", C.c_int64), ("dst_off", C.c_int64), ("stg_off", C.c_int64), ("row_bytes", C.c_int64),
                ("src_stride", C.c_int32), ("dst_stride", C.c_int32), ("nrows", C.c_int32),
                ("src_dev", C.c_int32), ("dst_rank", C.c_int32), ("dst_phys", C.c_int32), ("kind", C.c_int32),
                ("pad", C.c_int32)]


def lib():
    """Load libetc.so; fail loudly if it is missing (there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} not found: build it with `python -m paper_2607_04749_b200._build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(_LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.etc_init.restype = i32; L.etc_init.argtypes = [i32]
        L.etc_layout_create.restype = i32
        L.etc_layout_create.argtypes = [C.POINTER(_ModelDesc), C.POINTER(_ParallelCfg), C.POINTER(vp)]
        L.etc_layout_destroy.restype = None; L.etc_layout_destroy.argtypes = [vp]
        L.etc_layout_num_devices.restype = i32; L.etc_layout_num_devices.argtypes = [vp]
        L.etc_layout_num_pieces.restype = i64; L.etc_layout_num_pieces.argtypes = [vp]
        L.etc_layout_buffer_bytes.restype = i64; L.etc_layout_buffer_bytes.argtypes = [vp, i32, i32]
        L.etc_cost_matrix.restype = i32; L.etc_cost_matrix.argtypes = [vp, vp, vp, vp, vp, vp]
        L.etc_sketch.restype = i32; L.etc_sketch.argtypes = [vp, i32, i32, vp, i32, vp, vp, vp]
        L.etc_sketch_static.restype = i32; L.etc_sketch_static.argtypes = [vp, i32, i32, vp, vp, vp, vp]
        L.etc_defrag.restype = i32; L.etc_defrag.argtypes = [vp, i32, i32, i32, i32, vp, vp, vp, vp]
        L.etc_plan_create.restype = i32; L.etc_plan_create.argtypes = [vp, vp, vp, i32, C.POINTER(vp), vp]
        L.etc_plan_create_failed.restype = i32
        L.etc_plan_create_failed.argtypes = [vp, vp, vp, vp, i32, C.POINTER(vp), vp]
        L.etc_mask_failed.restype = i32; L.etc_mask_failed.argtypes = [vp, vp, i32, i32, i32, vp, vp]
        L.etc_mask_cross_dp.restype = i32; L.etc_mask_cross_dp.argtypes = [vp, vp, vp, vp]
        L.etc_plan_destroy.restype = None; L.etc_plan_destroy.argtypes = [vp]
        L.etc_plan_get_stats.restype = i32; L.etc_plan_get_stats.argtypes = [vp, C.POINTER(_PlanStats)]
        L.etc_plan_is_deferred.restype = i32; L.etc_plan_is_deferred.argtypes = [vp]
        L.etc_plan_get_traffic.restype = i32; L.etc_plan_get_traffic.argtypes = [vp, vp]
        L.etc_plan_get_slices.restype = i32; L.etc_plan_get_slices.argtypes = [vp, i32, vp]
        L.etc_plan_get_map.restype = i32; L.etc_plan_get_map.argtypes = [vp, vp]
        L.etc_plan_get_chunks.restype = i32; L.etc_plan_get_chunks.argtypes = [vp, i32, vp]
        L.etc_plan_get_fills.restype = i32; L.etc_plan_get_fills.argtypes = [vp, vp]
        L.etc_plan_validate.restype = i32; L.etc_plan_validate.argtypes = [vp, C.POINTER(i64), vp]
        L.etc_migrate.restype = i32; L.etc_migrate.argtypes = [vp, vp, vp, vp, vp]
        L.etc_migrate_phase.restype = i32; L.etc_migrate_phase.argtypes = [vp, vp, vp, vp, i32, vp]
        L.etc_plan_set_rounds.restype = i32; L.etc_plan_set_rounds.argtypes = [vp, i64, C.POINTER(i32), vp]
        L.etc_plan_get_round.restype = i32; L.etc_plan_get_round.argtypes = [vp, i32, C.POINTER(_RoundInfo)]
        L.etc_migrate_round.restype = i32; L.etc_migrate_round.argtypes = [vp, i32, vp, vp, vp, i32, vp]
        L.etc_upload_sources.restype = i32; L.etc_upload_sources.argtypes = [vp, vp, vp, i32, C.POINTER(i64), vp]
        L.etc_staging_bound.restype = i64; L.etc_staging_bound.argtypes = [vp, vp, i32]
        L.etc_migrate_state.restype = i32
        L.etc_migrate_state.argtypes = [C.POINTER(_ModelDesc), C.POINTER(_ParallelCfg), C.POINTER(_ParallelCfg), vp, vp, vp,
                                        i64, vp, i32, C.POINTER(vp), vp]
        L.etc_status_string.restype = C.c_char_p; L.etc_status_string.argtypes = [i32]
        L.etc_last_error_detail.restype = C.c_char_p
        L.etc_kernel_launches.restype = i64
        _lib = L
    return _lib


def _check(code):
    if code != 0:
        raise EtcError(code, lib().etc_last_error_detail().decode())


def init(device: int | None = None):
    """Bind the library to a CUDA device (default: torch's current device).  Raises without a GPU."""
    global _inited
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2607_04749_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    if device is None:
        device = torch.cuda.current_device()
    torch.cuda.init()
    _check(lib().etc_init(int(device)))
    _inited = True


def _ensure_init():
    if not _inited:
        init()


def _stream(stream=None) -> int:
    import torch
    return (stream or torch.cuda.current_stream()).cuda_stream


def kernel_launches() -> int:
    return int(lib().etc_kernel_launches())


class Layout:
    """Handle of an etc_layout (immutable)."""

    def __init__(self, handle, model, cfg):
        self.h, self.model, self.cfg = handle, dict(model), dict(cfg)
        self.n_dev = int(lib().etc_layout_num_devices(handle))
        self.n_pieces = int(lib().etc_layout_num_pieces(handle))

    def buffer_bytes(self, dev: int, kind: int) -> int:
        return int(lib().etc_layout_buffer_bytes(self.h, dev, kind))

    def kinds(self):
        return [k for k in range(4) if (self.model["kinds"] >> k) & 1]

    def total_bytes(self) -> int:
        return sum(self.buffer_bytes(d, k) for d in range(self.n_dev) for k in range(4))

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.etc_layout_destroy(self.h)
            self.h = None


def etc_layout_create(model: dict, cfg: dict) -> Layout:
    """(a1) include/etc.h etc_layout_create.  model: etc_inputs workload["model"] dict; cfg: {"tp","pp","dp","dist_opt"}."""
    _ensure_init()
    m, c = _model_struct(model), _cfg_struct(cfg)
    h = C.c_void_p()
    _check(lib().etc_layout_create(C.byref(m), C.byref(c), C.byref(h)))
    return Layout(h, model, cfg)


def etc_cost_matrix(old: Layout, new: Layout, stream=None, out=None):
    """(a2) -> (overlap [n_new][P], need [n_new], hold [P]) int64 CUDA tensors.  Asynchronous."""
    import torch
    P = max(old.n_dev, new.n_dev)
    if out is None:
        dev = torch.device("cuda", torch.cuda.current_device())
        out = (torch.empty((new.n_dev, P), dtype=torch.int64, device=dev),
               torch.empty(new.n_dev, dtype=torch.int64, device=dev), torch.empty(P, dtype=torch.int64, device=dev))
    ov, need, hold = out
    _check(lib().etc_cost_matrix(old.h, new.h, ov.data_ptr(), need.data_ptr(), hold.data_ptr(), _stream(stream)))
    return ov, need, hold


def etc_sketch(overlap, avail=None, method: int = ETC_SKETCH_AUTO, stream=None, out=None):
    """(a3) -> (device_map [n_new] int32, local_bytes [1] int64) CUDA tensors.  Asynchronous."""
    import torch
    _ensure_init()
    n_new, P = overlap.shape
    assert overlap.is_cuda and overlap.dtype == torch.int64 and overlap.is_contiguous()
    if out is None:
        out = (torch.empty(n_new, dtype=torch.int32, device=overlap.device),
               torch.empty(1, dtype=torch.int64, device=overlap.device))
    dm, lb = out
    av = 0
    if avail is not None:
        assert avail.is_cuda and avail.dtype == torch.uint8 and avail.numel() == P
        av = avail.data_ptr()
    _check(lib().etc_sketch(overlap.data_ptr(), n_new, P, av, method, dm.data_ptr(), lb.data_ptr(), _stream(stream)))
    return dm, lb


def etc_sketch_static(overlap, out, avail=None, stream=None):
    """(a3) etc_sketch for callers that must not allocate device memory (a trainer whose caching allocator already owns all
    free HBM, a recovery handler that must not stall on the allocator, a process with a fixed memory budget): the work area
    is a 28 KB array resident in libetc.so's device image, so this wrapper allocates nothing either — `out` =
    (device_map [n_new] int32, local_bytes [1] int64) must be passed in.  P <= ETC_SKETCH_STATIC_MAX_P (1024), else
    EtcError(ETC_ERR_WORKSPACE).  Same result as etc_sketch(method=ETC_SKETCH_HUNGARIAN).  All calls share the one work area:
    keep them on one stream (or order them); the first call on a device does a one-time address look-up, so make it at
    start-up.  Asynchronous; returns `out`."""
    import torch
    _ensure_init()
    n_new, P = overlap.shape
    assert overlap.is_cuda and overlap.dtype == torch.int64 and overlap.is_contiguous()
    dm, lb = out
    assert dm.is_cuda and dm.dtype == torch.int32 and dm.numel() >= n_new and lb.is_cuda and lb.dtype == torch.int64
    av = 0
    if avail is not None:
        assert avail.is_cuda and avail.dtype == torch.uint8 and avail.numel() == P
        av = avail.data_ptr()
    _check(lib().etc_sketch_static(overlap.data_ptr(), n_new, P, av, dm.data_ptr(), lb.data_ptr(), _stream(stream)))
    return dm, lb


def etc_defrag(device_map, pw: int, cw: int, devices_per_node: int, mode: int = ETC_DEFRAG_BOTH, want_ops: bool = True,
               stream=None):
    """(f1) include/etc.h etc_defrag.  device_map: CUDA int32 tensor [cw].  -> (out_map [cw] int32, n_ops [2] int32,
    ops [2][cw][2] int32 or None), all CUDA tensors.  Asynchronous."""
    import torch
    _ensure_init()
    assert device_map.is_cuda and device_map.dtype == torch.int32 and device_map.numel() == cw
    assert device_map.is_contiguous()
    out = torch.empty(cw, dtype=torch.int32, device=device_map.device)
    n_ops = torch.empty(2, dtype=torch.int32, device=device_map.device)
    ops = torch.full((2, cw, 2), -9, dtype=torch.int32, device=device_map.device) if want_ops else None
    _check(lib().etc_defrag(device_map.data_ptr(), pw, cw, devices_per_node, mode, out.data_ptr(),
                            ops.data_ptr() if want_ops else 0, n_ops.data_ptr(), _stream(stream)))
    return out, n_ops, ops


@dataclass
class PlanStats:
    staging_bytes: int
    local_bytes: int
    remote_bytes: int
    staged_bytes: int
    n_slices_local: int
    n_slices_staged: int
    n_chunks_local: int
    n_chunks_staged: int
    n_old: int
    n_new: int
    P: int
    flags: int
    fill_bytes: int = 0
    n_fills: int = 0

    @property
    def hbm_bytes(self) -> int:
        """Algorithmic HBM traffic of one etc_migrate: 1R+1W per local byte, 2R+2W per staged byte."""
        direct = self.local_bytes + self.remote_bytes - self.staged_bytes
        return 2 * direct + 4 * self.staged_bytes


class Plan:
    def __init__(self, handle, lazy: bool = False):
        self.h = handle
        self._stats = None
        if not lazy:
            self.stats                                    # read now (no wait: the plan was made the synchronising way)

    @property
    def stats(self) -> PlanStats:
        """etc_plan_get_stats; for an ETC_NO_SYNC plan the first access waits for the plan's kernels."""
        if self._stats is None:
            s = _PlanStats()
            _check(lib().etc_plan_get_stats(self.h, C.byref(s)))
            self._stats = PlanStats(**{n: int(getattr(s, n)) for n, _ in _PlanStats._fields_})
        return self._stats

    def traffic(self):
        import numpy as np
        P = self.stats.P
        T = np.zeros((P, P), np.int64)
        _check(lib().etc_plan_get_traffic(self.h, T.ctypes.data))
        return T

    def device_map(self):
        """the device map the plan was made for (host numpy int32 [n_new]); synchronous."""
        import numpy as np
        n = getattr(self, "n_new", None) or self.stats.n_new
        m = np.zeros(n, np.int32)
        _check(lib().etc_plan_get_map(self.h, m.ctypes.data))
        return m

    def slices(self, which: int):
        """which = 0 staged, 1 local -> numpy structured array of etc_slice records."""
        import numpy as np
        n = self.stats.n_slices_staged if which == 0 else self.stats.n_slices_local
        dt = np.dtype([(f, np.int64 if t is C.c_int64 else np.int32) for f, t in _Slice._fields_], align=True)
        assert dt.itemsize == C.sizeof(_Slice)
        arr = np.zeros(max(n, 1), dt)
        _check(lib().etc_plan_get_slices(self.h, which, arr.ctypes.data))
        return arr[:n]

    def chunks(self, which: int):
        """etc_plan_get_chunks: 0 staged / 1 local chunks in plan order, 2 / 3 the address-ordered launch lists."""
        import numpy as np
        st = self.stats
        n = st.n_chunks_local if which == 1 else (st.n_chunks_staged + st.n_chunks_local if which == 2 else st.n_chunks_staged)
        dt = np.dtype([("src_off", np.int64), ("dst_off", np.int64), ("stg_off", np.int64), ("src_stride", np.int32),
                       ("dst_stride", np.int32), ("row_bytes", np.int32), ("nrows", np.int32), ("src_buf", np.uint16),
                       ("dst_buf", np.uint16), ("vec", np.int16), ("staged", np.int16)])
        assert dt.itemsize == 48
        arr = np.zeros(max(n, 1), dt)
        _check(lib().etc_plan_get_chunks(self.h, which, arr.ctypes.data))
        return arr[:n]

    @property
    def deferred(self) -> bool:
        """etc_plan_is_deferred: True if ETC_NO_SYNC was honoured (counts still on the device; creation did not synchronise)."""
        r = lib().etc_plan_is_deferred(self.h)
        _check(min(r, 0))
        return r == 1

    def validate(self, stream=None) -> int:
        """device-side bounds check of every copy work item; returns the number of bad ones (0 for a sound plan)"""
        n = C.c_int64(-1)
        _check(lib().etc_plan_validate(self.h, C.byref(n), _stream(stream)))
        return int(n.value)

    def fills(self):
        """zero-fill descriptors (reading A31) as etc_slice records with src_dev = -1."""
        import numpy as np
        n = self.stats.n_fills
        dt = np.dtype([(f, np.int64 if t is C.c_int64 else np.int32) for f, t in _Slice._fields_], align=True)
        arr = np.zeros(max(n, 1), dt)
        _check(lib().etc_plan_get_fills(self.h, arr.ctypes.data))
        return arr[:n]

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.etc_plan_destroy(self.h)
            self.h = None


def etc_mask_failed(overlap, hold, failed, n_old: int, stream=None):
    """(f4) zero the failed old devices' columns of overlap [n_new][P] and entries of hold [P] in place.
    failed: CUDA uint8 tensor [n_old]."""
    import torch
    n_new, P = overlap.shape
    assert failed.is_cuda and failed.dtype == torch.uint8 and failed.numel() == n_old
    _check(lib().etc_mask_failed(overlap.data_ptr(), 0 if hold is None else hold.data_ptr(), n_new, n_old, P,
                                 failed.data_ptr(), _stream(stream)))
    return overlap, hold


def etc_mask_cross_dp(old: Layout, new: Layout, overlap, stream=None):
    """The paper's DP isolation (reading A5): zero the cross-DP cells of overlap [n_new][P] in place."""
    _check(lib().etc_mask_cross_dp(old.h, new.h, overlap.data_ptr(), _stream(stream)))
    return overlap


def etc_plan_create(old: Layout, new: Layout, device_map, flags: int = ETC_LOCAL_DIRECT, stream=None,
                    failed=None) -> Plan:
    """(a4) device_map: CUDA int32 tensor (e.g. from etc_sketch) or a host sequence.  Synchronises the stream once.
    failed (f4): optional [n_old] uint8 mask, CUDA tensor or host sequence (include/etc.h etc_plan_create_failed)."""
    import numpy as np
    import torch
    if isinstance(device_map, torch.Tensor):
        assert device_map.dtype == torch.int32 and device_map.numel() == new.n_dev and device_map.is_contiguous()
        keep = device_map
        ptr = device_map.data_ptr()
    else:
        keep = np.ascontiguousarray(device_map, np.int32)
        assert keep.shape == (new.n_dev,)
        ptr = keep.ctypes.data
    fptr, fkeep = None, None
    if failed is not None:
        if isinstance(failed, torch.Tensor):
            assert failed.dtype == torch.uint8 and failed.numel() == old.n_dev and failed.is_contiguous()
            fkeep = failed; fptr = failed.data_ptr()
        else:
            fkeep = np.ascontiguousarray(failed, np.uint8)
            assert fkeep.shape == (old.n_dev,)
            fptr = fkeep.ctypes.data
    h = C.c_void_p()
    _check(lib().etc_plan_create_failed(old.h, new.h, ptr, fptr, flags, C.byref(h), _stream(stream)))
    del keep, fkeep
    p = Plan(h, lazy=bool(flags & ETC_NO_SYNC))
    p.n_old, p.n_new = old.n_dev, new.n_dev
    return p


def etc_staging_bound(old: Layout, new: Layout, flags: int = ETC_LOCAL_DIRECT) -> int:
    """include/etc.h etc_staging_bound: staging bytes that suffice for ANY device map between the two layouts."""
    n = int(lib().etc_staging_bound(old.h, new.h, flags))
    if n < 0:
        raise EtcError(n)
    return n


def _model_struct(model: dict) -> "_ModelDesc":
    return _ModelDesc(style=model["style"], n_layers=model["n_layers"], hidden=model["hidden"],
                      n_q_heads=model["n_q_heads"], n_kv_heads=model["n_kv_heads"], head_dim=model["head_dim"],
                      ffn_hidden=model["ffn_hidden"], vocab=model["vocab"], max_pos=model["max_pos"],
                      tied_embeddings=model["tied"], param_dtype=model["param_bytes"], kinds=model["kinds"],
                      qkv_order=model.get("qkv_order", 0))


def _cfg_struct(cfg: dict) -> "_ParallelCfg":
    return _ParallelCfg(tp=cfg["tp"], pp=cfg["pp"], dp=cfg["dp"], dist_opt=cfg.get("dist_opt", 0),
                        pp_first=cfg.get("pp_first", 0), pp_last=cfg.get("pp_last", 0),
                        dist_opt_align=cfg.get("dist_opt_align", 0), vocab_divisor=cfg.get("vocab_divisor", 0))


class MigrateState:
    """Pre-marshalled arguments of etc_migrate_state for one (model, old cfg, new cfg, buffers): calling it is ONE
    C-ABI call that enqueues the whole path (a1)-(a6) without a host synchronisation."""

    def __init__(self, model: dict, old_cfg: dict, new_cfg: dict, src_bufs, dst_bufs, staging, flags: int = ETC_LOCAL_DIRECT,
                 avail=None):
        _ensure_init()
        self.m, self.oc, self.nc = _model_struct(model), _cfg_struct(old_cfg), _cfg_struct(new_cfg)
        n_old = old_cfg["tp"] * old_cfg["pp"] * old_cfg["dp"]
        n_new = new_cfg["tp"] * new_cfg["pp"] * new_cfg["dp"]
        self.n_old, self.n_new = n_old, n_new
        self.src = _ptr_table(src_bufs, n_old) if isinstance(src_bufs, dict) else src_bufs
        self.dst = _ptr_table(dst_bufs, n_new) if isinstance(dst_bufs, dict) else dst_bufs
        self.keep = (src_bufs, dst_bufs, staging, avail)
        self.stg = staging.data_ptr() if staging is not None and staging.numel() else 0
        self.stg_bytes = staging.numel() * staging.element_size() if staging is not None else 0
        self.avail = avail.data_ptr() if avail is not None else 0
        self.flags = flags

    def __call__(self, stream=None, want_plan: bool = False):
        h = C.c_void_p()
        _check(lib().etc_migrate_state(C.byref(self.m), C.byref(self.oc), C.byref(self.nc), self.src, self.dst, self.stg,
                                       self.stg_bytes, self.avail, self.flags, C.byref(h) if want_plan else None,
                                       _stream(stream)))
        if want_plan:
            p = Plan(h, lazy=True)
            p.n_old, p.n_new = self.n_old, self.n_new
            return p
        return None


def etc_migrate_state(model: dict, old_cfg: dict, new_cfg: dict, src_bufs, dst_bufs, staging, flags: int = ETC_LOCAL_DIRECT,
                      avail=None, stream=None, want_plan: bool = True):
    """include/etc.h etc_migrate_state: the whole path in one call.  Returns the plan (lazy statistics) or None."""
    return MigrateState(model, old_cfg, new_cfg, src_bufs, dst_bufs, staging, flags, avail)(stream, want_plan)


def _ptr_table(bufs, n_dev):
    tab = (C.c_void_p * (n_dev * 4))()
    for (dev, kind), t in bufs.items():
        if t is not None and t.numel() > 0:
            tab[dev * 4 + kind] = t.data_ptr()
    return tab


def etc_migrate(plan: Plan, src_bufs: dict, dst_bufs: dict, staging, phases: int = ETC_PHASE_ALL, stream=None):
    """(a5,a6) src_bufs {(old_dev, kind): CUDA tensor}, dst_bufs {(new_rank, kind): CUDA tensor}, staging: CUDA tensor
    of at least plan.stats.staging_bytes bytes (or None).  Asynchronous; no allocation."""
    n_old, n_new = getattr(plan, "n_old", None), getattr(plan, "n_new", None)
    if n_old is None:
        n_old, n_new = plan.stats.n_old, plan.stats.n_new
    if isinstance(src_bufs, dict):
        src_bufs = _ptr_table(src_bufs, n_old)
    if isinstance(dst_bufs, dict):
        dst_bufs = _ptr_table(dst_bufs, n_new)
    sp = 0
    if staging is not None and staging.numel() > 0:
        if plan._stats is not None:                   # a lazy (ETC_NO_SYNC) plan: the caller sized it by etc_staging_bound
            assert staging.numel() * staging.element_size() >= plan._stats.staging_bytes
        sp = staging.data_ptr()
    _check(lib().etc_migrate_phase(plan.h, src_bufs, dst_bufs, sp, phases, _stream(stream)))


def etc_upload_sources(plan: Plan, h_src_bufs, d_src_bufs, only_kind: int = -1, stream=None) -> int:
    """Host-resident old shards: copy exactly the regions the plan reads from the pinned host buffers to the same offsets
    of the device buffers (include/etc.h etc_upload_sources).  Dicts {(old_dev, kind): tensor} or pointer tables.
    Returns the bytes enqueued."""
    st = plan.stats
    if isinstance(h_src_bufs, dict):
        h_src_bufs = _ptr_table(h_src_bufs, st.n_old)
    if isinstance(d_src_bufs, dict):
        d_src_bufs = _ptr_table(d_src_bufs, st.n_old)
    n = C.c_int64(0)
    _check(lib().etc_upload_sources(plan.h, h_src_bufs, d_src_bufs, only_kind, C.byref(n), _stream(stream)))
    return int(n.value)


@dataclass
class RoundInfo:
    kind: int
    sub: int
    n_sub: int
    staging_bytes: int
    staged_bytes: int
    local_bytes: int
    n_chunks_staged: int
    n_chunks_local: int

    @property
    def hbm_bytes(self) -> int:
        return 2 * self.local_bytes + 4 * self.staged_bytes


def etc_plan_set_rounds(plan: Plan, max_staging_bytes: int, stream=None):
    """(f2) include/etc.h etc_plan_set_rounds -> [RoundInfo].  The plan must have been created with ETC_KIND_MAJOR."""
    n = C.c_int32()
    _check(lib().etc_plan_set_rounds(plan.h, int(max_staging_bytes), C.byref(n), _stream(stream)))
    out = []
    for r in range(n.value):
        info = _RoundInfo()
        _check(lib().etc_plan_get_round(plan.h, r, C.byref(info)))
        out.append(RoundInfo(**{f: int(getattr(info, f)) for f, _ in _RoundInfo._fields_ if f != "pad"}))
    plan.rounds = out
    return out


def etc_migrate_round(plan: Plan, rnd: int, src_bufs, dst_bufs, staging, phases: int = ETC_PHASE_ALL, stream=None):
    """(f2) one round; only the buffers of the round's kind need to exist in src_bufs / dst_bufs."""
    st = plan.stats
    if isinstance(src_bufs, dict):
        src_bufs = _ptr_table(src_bufs, st.n_old)
    if isinstance(dst_bufs, dict):
        dst_bufs = _ptr_table(dst_bufs, st.n_new)
    sp = 0
    if staging is not None and staging.numel() > 0:
        assert staging.numel() * staging.element_size() >= plan.rounds[rnd].staging_bytes
        sp = staging.data_ptr()
    _check(lib().etc_migrate_round(plan.h, rnd, src_bufs, dst_bufs, sp, phases, _stream(stream)))


def pointer_tables(plan: Plan, src_bufs: dict, dst_bufs: dict):
    """Pre-marshalled pointer tables (avoids rebuilding them on every etc_migrate call)."""
    return _ptr_table(src_bufs, plan.stats.n_old), _ptr_table(dst_bufs, plan.stats.n_new)


def alloc_buffers(layout: Layout, device=None, fill=None):
    """{(dev, kind): uint8 CUDA tensor of etc_layout_buffer_bytes} for every non-empty buffer."""
    import torch
    device = device or torch.device("cuda", torch.cuda.current_device())
    out = {}
    for d in range(layout.n_dev):
        for k in range(4):
            n = layout.buffer_bytes(d, k)
            if n > 0:
                out[(d, k)] = torch.empty(n, dtype=torch.uint8, device=device) if fill is None else \
                    torch.full((n,), fill, dtype=torch.uint8, device=device)
    return out
