"""CPU-side checks of the C-ABI boundary: libetc.so loads and exports every symbol include/etc.h declares; argument
validation that needs no GPU.  (No compute calls here.)"""
from __future__ import annotations
import ctypes as C
import os
import re
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_04749_b200 import _build, binding
    _build.build()
    return binding.lib()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "etc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(etc_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_functions()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), f"libetc.so does not export {n}"
    from paper_2607_04749_b200 import EXPORTED_SYMBOLS
    assert sorted(EXPORTED_SYMBOLS) == names


def test_status_strings(lib):
    assert lib.etc_status_string(0) == b"ETC_OK"
    for code, name in [(-1, b"ETC_ERR_INVALID_ARG"), (-2, b"ETC_ERR_INDIVISIBLE"), (-3, b"ETC_ERR_MISMATCH"),
                       (-4, b"ETC_ERR_BAD_MAP"), (-5, b"ETC_ERR_WORKSPACE"), (-6, b"ETC_ERR_UNSUPPORTED"),
                       (-7, b"ETC_ERR_CUDA")]:
        assert lib.etc_status_string(code) == name


def test_layout_validation_without_gpu(lib):
    """Validation errors are reported before any CUDA call (PAPER.md:277 divisibility; reading A10)."""
    from paper_2607_04749_b200.binding import _ModelDesc, _ParallelCfg
    m = _ModelDesc(style=0, n_layers=4, hidden=12, n_q_heads=2, n_kv_heads=2, head_dim=6, ffn_hidden=28, vocab=20,
                   max_pos=0, tied_embeddings=1, param_dtype=2, kinds=15)
    h = C.c_void_p()
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(1, 3, 1, 0)), C.byref(h)) == -2   # layers % pp
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(4, 1, 1, 0)), C.byref(h)) == -6   # tp > kv heads
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(0, 1, 1, 0)), C.byref(h)) == -1
    assert lib.etc_layout_create(None, C.byref(_ParallelCfg(1, 1, 1, 0)), C.byref(h)) == -1
    # uneven pipeline splits (f3, reading A27): validated on the host as well
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(1, 3, 1, 0, 1, 0)), C.byref(h)) == -2   # 3 layers / 2 stages
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(1, 2, 1, 0, 1, 1)), C.byref(h)) == -2   # 2 layers unassigned
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(1, 1, 1, 0, 4, 0)), C.byref(h)) == -1   # pp = 1
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(1, 2, 1, 0, -1, 0)), C.byref(h)) == -1
    m.param_dtype = 3
    assert lib.etc_layout_create(C.byref(m), C.byref(_ParallelCfg(1, 1, 1, 0)), C.byref(h)) == -1
    assert h.value is None


def test_one_call_primitive_validates_before_any_cuda_call(lib):
    """etc_migrate_state / etc_staging_bound / etc_plan_create reject bad arguments on the host."""
    from paper_2607_04749_b200.binding import _ModelDesc, _ParallelCfg
    m = _ModelDesc(style=0, n_layers=4, hidden=12, n_q_heads=2, n_kv_heads=2, head_dim=6, ffn_hidden=28, vocab=20,
                   max_pos=0, tied_embeddings=1, param_dtype=2, kinds=15)
    c = _ParallelCfg(1, 1, 1, 0)
    tab = (C.c_void_p * 4)()
    h = C.c_void_p()
    args = lambda **kw: [kw.get("m", C.byref(m)), kw.get("oc", C.byref(c)), kw.get("nc", C.byref(c)), kw.get("src", tab),
                         kw.get("dst", tab), None, kw.get("stg_bytes", 0), None, kw.get("flags", 0), C.byref(h), None]
    assert lib.etc_migrate_state(*args(m=None)) == -1
    assert lib.etc_migrate_state(*args(src=None)) == -1
    assert lib.etc_migrate_state(*args(stg_bytes=-1)) == -1
    assert lib.etc_migrate_state(*args(flags=2)) == -1            # ETC_KIND_MAJOR is for rounds, not for the one-call path
    assert lib.etc_migrate_state(*args(flags=8)) == -1            # ETC_NO_SYNC is implied, not a caller's flag here
    assert lib.etc_migrate_state(*args(nc=C.byref(_ParallelCfg(1, 3, 1, 0)))) == -2      # layers % pp
    assert h.value is None
    assert lib.etc_staging_bound(None, None, 0) == -1
    assert lib.etc_plan_create(None, None, None, 0, C.byref(h), None) == -1


def test_static_sketch_and_deferred_query_validate_on_the_host(lib):
    """etc_sketch_static refuses bad arguments and sizes beyond its resident work area before any CUDA call (so this runs
    without a GPU), with a readable text in etc_last_error_detail; the header's constants match the library's array
    (a static_assert in sketch.cu ties them to the kernel's row format); etc_plan_is_deferred(NULL) is an error."""
    src = open(os.path.join(ROOT, "include", "etc.h")).read()
    max_p = int(re.search(r"#define ETC_SKETCH_STATIC_MAX_P (\d+)", src).group(1))
    nbytes = int(re.search(r"#define ETC_SKETCH_STATIC_SCRATCH_BYTES (\d+)", src).group(1))
    from paper_2607_04749_b200 import ETC_SKETCH_STATIC_MAX_P, ETC_SKETCH_STATIC_SCRATCH_BYTES
    assert (max_p, nbytes) == (ETC_SKETCH_STATIC_MAX_P, ETC_SKETCH_STATIC_SCRATCH_BYTES) == (1024, 1024 * 28)
    buf = (C.c_int64 * 4)()
    p = C.addressof(buf)                                          # never dereferenced: every call below fails first
    assert lib.etc_sketch_static(None, 2, 4, None, p, p, None) == -1
    assert lib.etc_sketch_static(p, 2, 4, None, None, p, None) == -1
    assert lib.etc_sketch_static(p, 0, 4, None, p, p, None) == -1
    assert lib.etc_sketch_static(p, 5, 4, None, p, p, None) == -1            # more rows than columns
    assert lib.etc_sketch_static(p, 2, max_p + 1, None, p, p, None) == -5    # ETC_ERR_WORKSPACE
    detail = lib.etc_last_error_detail().decode()
    assert "ETC_SKETCH_STATIC_MAX_P" in detail and str(max_p + 1) in detail and "etc_sketch" in detail
    assert lib.etc_sketch_static(None, 2, 4, None, p, p, None) == -1 and lib.etc_last_error_detail() == b""   # cleared per call
    assert lib.etc_plan_is_deferred(None) == -1


def test_product_path_has_no_oracle_or_cpu_fallback():
    """The package must not import the oracle, and must fail loudly without a CUDA device."""
    import torch
    import paper_2607_04749_b200 as E
    pkg = os.path.join(ROOT, "paper_2607_04749_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):
            E.etc_layout_create(dict(style=0, n_layers=2, hidden=8, n_q_heads=2, n_kv_heads=2, head_dim=4,
                                     ffn_hidden=16, vocab=8, max_pos=0, tied=0, param_bytes=2, kinds=15),
                                dict(tp=1, pp=1, dp=1, dist_opt=0))
