"""-m "not gpu": pins of the oracle's layout variants (f3): uneven pipeline splits (reading A27, PAPER.md:277 requires
divisibility; Megatron-LM's --decoder-first/last-pipeline-num-layers) against hand-computed values, the layer-unit cost
formula of PAPER.md:106, and the whole P2-P10 battery on swept uneven reconfigurations."""
from __future__ import annotations
import numpy as np
import pytest

from etc_inputs import tiny_models
from etc_inputs.workloads import STYLE_GPT
from oracle import oracle as O
from helpers import read_golden
from test_oracle_pins import _check_reconfiguration

TINY = dict(tiny_models())
GOLD = read_golden("uneven_pp_handcomputed.txt")


def _cfg(tp, pp, dp, dist_opt=0, first=0, last=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt, pp_first=first, pp_last=last)


def _layer_model(n_layers):
    return dict(style=STYLE_GPT, n_layers=n_layers, hidden=8, n_q_heads=2, n_kv_heads=2, head_dim=4, ffn_hidden=16,
                vocab=8, max_pos=4, tied=0, param_bytes=2, kinds=0b1111)


@pytest.mark.parametrize("row", [r for r in GOLD if r[0] == "range"], ids=lambda r: "-".join(r[1:5]))
def test_stage_layer_ranges(row):
    """Which layers a stage holds, read back through global_of (TP=DP=1: device = stage)."""
    n_layers, pp, first, last = map(int, row[1:5])
    begins = [int(x) for x in row[6:]]
    model = _layer_model(n_layers)
    L = O.Layout(model, _cfg(1, pp, 1, 0, first, last))
    lts = O.logical_tensors(model)
    for s in range(pp):
        lt, _, _, _ = L.global_of(s, 0)
        layers = sorted({lts[t][4] for t in np.unique(lt) if lts[t][3] == 1})
        assert layers == list(range(begins[s], begins[s + 1])), (s, layers)


@pytest.mark.parametrize("row", [r for r in GOLD if r[0] == "elems"], ids=lambda r: "-".join(r[1:5]))
def test_device_element_counts(row):
    name, pp, first, last = row[1], int(row[2]), int(row[3]), int(row[4])
    L = O.Layout(TINY[name], _cfg(1, pp, 1, 0, first, last))
    assert [L.buffer_elems(d, 0) for d in range(pp)] == [int(x) for x in row[6:]]


def test_uneven_cost_matrix_in_layer_units():
    gold = np.array([[int(x) for x in r[1:]] for r in GOLD if r[0] == "cost"])
    model = _layer_model(16)
    old, new = O.Layout(model, _cfg(1, 4, 1)), O.Layout(model, _cfg(1, 3, 1, 0, 6, 4))
    ov, need, hold = O.overlap(old, new, only_layers=True)
    per_layer = hold[0] // 4
    assert hold[0] % 4 == 0 and ((need[:, None] - ov) % per_layer == 0).all()
    assert np.array_equal((need[:, None] - ov)[:, :4] // per_layer, gold)


def test_invalid_uneven_splits():
    m = TINY["gpt_t"]                                            # 4 layers
    for cfg, code in [(_cfg(1, 3, 1, 0, 1, 0), -2),              # 3 layers over 2 stages
                      (_cfg(1, 2, 1, 0, 1, 1), -2),              # 2 layers unassigned
                      (_cfg(1, 3, 1, 0, 2, 2), -2),              # nothing left for the middle stage
                      (_cfg(1, 1, 1, 0, 4, 0), -1),              # pp = 1 cannot be uneven
                      (_cfg(1, 2, 1, 0, -1, 0), -1)]:
        with pytest.raises(O.OracleError) as e:
            O.Layout(m, cfg)
        assert e.value.code == code, cfg
    O.Layout(m, _cfg(1, 2, 1, 0, 4 - 1, 1))                      # both fixed and consistent
    O.Layout(m, _cfg(1, 2, 1, 0, 2, 0))                          # same as the even split
    a, b = O.Layout(m, _cfg(2, 2, 2, 1, 2, 0)), O.Layout(m, _cfg(2, 2, 2, 1))
    assert all(a.buffer_elems(d, k) == b.buffer_elems(d, k) for d in range(8) for k in range(4))


def test_uneven_reconfigurations_full_battery():
    """P2-P5, P8-P10 (test_oracle_pins._check_reconfiguration) on reconfigurations into, out of and between uneven
    pipeline splits, with TP / DP / dist-opt changes, tied and untied, both styles."""
    cases = [("gpt_t", _cfg(1, 2, 1), _cfg(1, 3, 1, 0, 2, 0)),
             ("gpt_t", _cfg(2, 3, 1, 0, 0, 2), _cfg(1, 2, 2, 1, 1, 3)),
             ("gpt_np", _cfg(2, 2, 2, 1, 3, 1), _cfg(1, 4, 1)),
             ("llama_u", _cfg(2, 3, 1, 0, 2, 0), _cfg(1, 2, 2, 0, 3, 0)),
             ("llama_u", _cfg(1, 4, 2), _cfg(2, 3, 1, 0, 1, 1)),
             ("gpt_t", _cfg(1, 3, 2, 1, 1, 1), _cfg(2, 3, 1, 0, 2, 1))]
    rng = np.random.default_rng(3)
    for i, (name, a, b) in enumerate(cases):
        assert _check_reconfiguration(TINY[name], a, b, 900 + i)
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        dm = rng.permutation(max(na, nb))[:nb].astype(np.int32)
        assert _check_reconfiguration(TINY[name], a, b, 950 + i, device_map=dm)


# ---------------------------------------------------------------------------------------------- A28: aligned dist-opt
GOLD_ALIGN = read_golden("distopt_align_handcomputed.txt")


def _cfga(tp, pp, dp, align, dist_opt=1):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt, dist_opt_align=align)


@pytest.mark.parametrize("row", GOLD_ALIGN, ids=lambda r: "-".join(r[1:7]))
def test_aligned_distopt_ranges_handcomputed(row):
    name, tp, pp, dp, align = row[1], int(row[2]), int(row[3]), int(row[4]), int(row[5])
    L = O.Layout(TINY[name], _cfga(tp, pp, dp, align))
    got = [L.buffer_elems(0 + tp * d, 1) for d in range(dp)]            # device id = r + tp*(d + dp*s), r = s = 0
    assert got == [int(x) for x in row[7:]]
    # PARAM stays replicated (BASELINE.json config 4), M and V follow MASTER
    assert len({L.buffer_elems(tp * d, 0) for d in range(dp)}) == 1
    assert all(L.buffer_elems(tp * d, 2) == got[d] and L.buffer_elems(tp * d, 3) == got[d] for d in range(dp))


def test_aligned_distopt_invariants():
    """Every shard boundary is a multiple of the alignment, shards tile the local space exactly once, and alignment
    changes nothing when the kind is not DP-sharded."""
    for name, model in TINY.items():
        for tp, pp, dp, align in [(1, 2, 2, 16), (2, 1, 4, 8), (1, 1, 3, 100), (2, 2, 2, 7)]:
            try:
                L = O.Layout(model, _cfga(tp, pp, dp, align))
                R = O.Layout(model, _cfga(tp, pp, dp, align, dist_opt=0))
            except O.OracleError:
                continue
            for s in range(pp):
                for r in range(tp):
                    sizes = [L.buffer_elems(r + tp * (d + dp * s), 2) for d in range(dp)]
                    assert sum(sizes) == R.buffer_elems(r + tp * dp * s, 2)
                    full = [x for x in sizes if x and x != sizes[0]]
                    assert sizes[0] % align == 0 or sum(sizes) == sizes[0]
                    assert len(full) <= 1                                  # only one ragged shard
                    lts = [L.global_of(r + tp * (d + dp * s), 2) for d in range(dp) if sizes[d]]
                    ref = R.global_of(r + tp * dp * s, 2)
                    for j in range(4):
                        assert np.array_equal(np.concatenate([x[j] for x in lts]), ref[j])
    with pytest.raises(O.OracleError):
        O.Layout(TINY["gpt_t"], _cfga(1, 1, 2, -4))


def test_aligned_distopt_full_battery():
    """P2-P5, P8-P10 on reconfigurations between differently aligned distributed-optimizer layouts."""
    cases = [("gpt_t", _cfga(1, 1, 4, 128), _cfga(2, 1, 2, 64)),
             ("gpt_t", _cfga(2, 2, 2, 32), _cfga(1, 2, 2, 0, dist_opt=0)),
             ("gpt_np", _cfga(1, 2, 2, 0), _cfga(2, 2, 2, 48)),
             ("llama_u", _cfga(2, 1, 4, 24), _cfga(1, 2, 3, 40)),
             ("llama_t", _cfga(1, 2, 3, 1000), _cfga(2, 2, 2, 8))]
    rng = np.random.default_rng(11)
    for i, (name, a, b) in enumerate(cases):
        assert _check_reconfiguration(TINY[name], a, b, 1200 + i)
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        dm = rng.permutation(max(na, nb))[:nb].astype(np.int32)
        assert _check_reconfiguration(TINY[name], a, b, 1250 + i, device_map=dm)
