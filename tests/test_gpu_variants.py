"""-m gpu parity of the layout variants (f3): uneven pipeline splits (reading A27) through the whole CUDA path against
the element-wise oracle."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import tiny_models, workload
from oracle import oracle as O
from test_gpu_parity import _check_migration


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _cfg(tp, pp, dp, dist_opt=0, first=0, last=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt, pp_first=first, pp_last=last)


def test_uneven_pipeline_tiny(E):
    T = dict(tiny_models())
    cases = [("gpt_t", _cfg(1, 2, 1), _cfg(1, 3, 1, 0, 2, 0)),
             ("gpt_t", _cfg(2, 3, 1, 0, 0, 2), _cfg(1, 2, 2, 1, 1, 3)),
             ("gpt_np", _cfg(2, 2, 2, 1, 3, 1), _cfg(1, 4, 1)),
             ("llama_u", _cfg(2, 3, 1, 0, 2, 0), _cfg(1, 2, 2, 0, 3, 0)),
             ("llama_u", _cfg(1, 4, 2), _cfg(2, 3, 1, 0, 1, 1)),
             ("gpt_t", _cfg(1, 3, 2, 1, 1, 1), _cfg(2, 3, 1, 0, 2, 1))]
    rng = np.random.default_rng(31)
    for i, (name, a, b) in enumerate(cases):
        for flags in (0, 3):
            _check_migration(E, T[name], a, b, 700 + i, flags=flags)
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        _check_migration(E, T[name], a, b, 750 + i, device_map=rng.permutation(max(na, nb))[:nb].astype(np.int32))


def test_uneven_pipeline_scaled_preemption(E):
    """s3's model (12 layers) pre-empted from TP4 PP4 (16 devices) to TP4 PP3 with an uneven 5/4/3 split: more layers on
    the first stage, fewer on the last (which also holds the tied embedding replica)."""
    w = workload("s3")
    new = _cfg(4, 3, 1, 0, 5, 3)
    for flags in (0, 1):
        g = _check_migration(E, w["model"], w["old"], new, w["seed"], flags=flags)
    assert g["plan"].stats.remote_bytes > 0


def test_uneven_validation_codes_match_oracle(E):
    m = dict(tiny_models())["gpt_t"]
    for cfg in (_cfg(1, 3, 1, 0, 1, 0), _cfg(1, 2, 1, 0, 1, 1), _cfg(1, 1, 1, 0, 4, 0), _cfg(8, 3, 1, 0, 2, 0)):
        with pytest.raises(O.OracleError) as oe:
            O.Layout(m, cfg)
        with pytest.raises(E.EtcError) as ge:
            E.etc_layout_create(m, cfg)
        assert ge.value.code == oe.value.code, cfg


# ---------------------------------------------------------------------------------------------- A28: aligned dist-opt
def _cfga(tp, pp, dp, align, dist_opt=1):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt, dist_opt_align=align)


def test_aligned_distopt_tiny(E):
    T = dict(tiny_models())
    cases = [("gpt_t", _cfga(1, 1, 4, 128), _cfga(2, 1, 2, 64)),
             ("gpt_t", _cfga(2, 2, 2, 32), _cfga(1, 2, 2, 0, dist_opt=0)),
             ("gpt_np", _cfga(1, 2, 2, 0), _cfga(2, 2, 2, 48)),
             ("llama_u", _cfga(2, 1, 4, 24), _cfga(1, 2, 3, 40)),
             ("llama_t", _cfga(1, 2, 3, 1000), _cfga(2, 2, 2, 8)),
             ("gpt_t", _cfga(1, 1, 4, 1024), _cfga(1, 1, 4, 128))]         # a DP rank that holds nothing
    rng = np.random.default_rng(41)
    for i, (name, a, b) in enumerate(cases):
        for flags in (0, 3):
            _check_migration(E, T[name], a, b, 800 + i, flags=flags)
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        _check_migration(E, T[name], a, b, 850 + i, device_map=rng.permutation(max(na, nb))[:nb].astype(np.int32))
    la = E.etc_layout_create(T["gpt_t"], _cfga(1, 1, 4, 128))
    assert [la.buffer_bytes(d, 1) for d in range(4)] == [640 * 4, 640 * 4, 640 * 4, 592 * 4]   # tests/golden, hand-computed
    with pytest.raises(E.EtcError) as ge:
        E.etc_layout_create(T["gpt_t"], _cfga(1, 1, 2, -4))
    assert ge.value.code == -1


def test_aligned_distopt_scaled_c4(E):
    """s4 (config 4's reconfiguration, TP2 PP4 DP2 -> TP4 PP2 DP4, distributed optimizer on both sides) with 128-element
    aligned DP shards on the old side and 256-element aligned shards on the new side."""
    w = workload("s4")
    old, new = dict(w["old"], dist_opt_align=128), dict(w["new"], dist_opt_align=256)
    for flags in (0, 1):
        g = _check_migration(E, w["model"], old, new, w["seed"], flags=flags)
    assert g["plan"].stats.remote_bytes > 0
