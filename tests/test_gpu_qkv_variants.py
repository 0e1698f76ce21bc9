"""-m gpu parity of the fused-QKV layout variants (f3c, f3d): [Q;K;V] block row order (reading A29) and KV-head
replication when tp > n_kv (reading A30) through the whole CUDA path against the element-wise oracle: cost matrices,
sketch objective, traffic matrix, slice coverage and every destination buffer bit for bit."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload
from etc_inputs.workloads import STYLE_GPT, STYLE_LLAMA
from oracle import oracle as O
from test_gpu_parity import _check_migration


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _model(style=STYLE_LLAMA, order=0, n_q=4, n_kv=2, d=2, layers=2, hidden=8, tied=0, kinds=0b1111):
    return dict(style=style, n_layers=layers, hidden=hidden, n_q_heads=n_q, n_kv_heads=n_kv, head_dim=d, ffn_hidden=16,
                vocab=8, max_pos=4 if style == STYLE_GPT else 0, tied=tied, param_bytes=2, kinds=kinds, qkv_order=order)


def _cfg(tp, pp=1, dp=1, dist_opt=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt)


CASES = [(_model(STYLE_LLAMA, 0), _cfg(2), _cfg(4)), (_model(STYLE_LLAMA, 0), _cfg(4), _cfg(1, 2)),
         (_model(STYLE_LLAMA, 1), _cfg(1, 2), _cfg(2)), (_model(STYLE_LLAMA, 1), _cfg(4), _cfg(2, 1, 2)),
         (_model(STYLE_GPT, 1, tied=1), _cfg(4, 2), _cfg(2, 1, 2, 1)),
         (_model(STYLE_GPT, 0, tied=1), _cfg(2, 1, 2, 1), _cfg(4, 2)),
         (_model(STYLE_LLAMA, 0, n_q=8, n_kv=2, hidden=16), _cfg(8), _cfg(4, 1, 2, 1)),
         (_model(STYLE_LLAMA, 1, n_q=8, n_kv=2, hidden=16), _cfg(4, 1, 2, 1), _cfg(8)),
         (_model(STYLE_LLAMA, 0, n_q=4, n_kv=1), _cfg(4), _cfg(2, 2)),
         (_model(STYLE_LLAMA, 1, n_q=8, n_kv=2, hidden=16), _cfg(8, 1, 2, 1), _cfg(4, 2, 2, 1)),   # dist-opt cuts through Q/K/V blocks
         (_model(STYLE_GPT, 0, n_q=8, n_kv=2, hidden=16), _cfg(4, 2, 2), _cfg(8, 1, 2)),           # DP round-robin x TP round-robin
         (_model(STYLE_GPT, 1, n_q=8, n_kv=2, hidden=16, tied=1), _cfg(8, 2), _cfg(8, 1, 2))]


@pytest.mark.parametrize("i", range(len(CASES)))
def test_qkv_variants_tiny(E, i):
    m, a, b = CASES[i]
    rng = np.random.default_rng(900 + i)
    for flags in (0, 3):
        _check_migration(E, m, a, b, 1500 + i, flags=flags)
    na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
    for rep in range(2):
        dm = rng.permutation(max(na, nb))[:nb].astype(np.int32)
        _check_migration(E, m, a, b, 1550 + i, device_map=dm)


def test_qkv_shard_rows_through_the_slice_table(E):
    """tests/golden/qkv_variants_handcomputed.txt through the CUDA path: migrate a TP1 layout whose QKV rows carry their
    own row index into TP4 (KV-replicated) and read the hand-computed rows back from the new shards."""
    from helpers import read_golden
    for g in read_golden("qkv_variants_handcomputed.txt"):
        order, tp, r = int(g[1]), int(g[2]), int(g[3])
        want = [int(x) for x in g[5:]]
        m = _model(STYLE_LLAMA, order, kinds=0b0010)
        old, new = E.etc_layout_create(m, _cfg(1)), E.etc_layout_create(m, _cfg(tp))
        # local order at TP1: word_embeddings (8x8), layer 0: ln1 (8), qkv (16x8) ...
        n_el = old.buffer_bytes(0, 1) // 4
        src = torch.zeros(n_el, dtype=torch.int32, device="cuda")
        qkv0 = 8 * 8 + 8
        src[qkv0:qkv0 + 16 * 8] = torch.arange(16, dtype=torch.int32, device="cuda").repeat_interleave(8) + 100
        plan = E.etc_plan_create(old, new, torch.arange(tp, dtype=torch.int32, device="cuda"))
        dst = E.alloc_buffers(new, fill=0)
        stg = torch.empty(max(plan.stats.staging_bytes, 16), dtype=torch.uint8, device="cuda")
        E.etc_migrate(plan, {(0, 1): src.view(torch.uint8)}, dst, stg)
        torch.cuda.synchronize()
        got = dst[(r, 1)].view(torch.int32).cpu().numpy()
        pre = (8 // tp) * 8 + 8                              # word_embeddings (8/tp rows x 8), ln1.weight (8)
        rows = got[pre:pre + len(want) * 8].reshape(len(want), 8)
        assert (rows == (np.asarray(want)[:, None] + 100)).all(), (order, tp, r)


def test_qkv_validation_codes_match_oracle(E):
    for model, cfg in [(_model(n_q=8, n_kv=4, hidden=24), _cfg(3)), (_model(n_q=8, n_kv=2), _cfg(6)),
                       (_model(n_q=6, n_kv=2, hidden=12), _cfg(4)), (_model(order=2), _cfg(1))]:
        with pytest.raises(O.OracleError) as oe:
            O.Layout(model, cfg)
        with pytest.raises(E.EtcError) as ge:
            E.etc_layout_create(model, cfg)
        assert ge.value.code == oe.value.code, (model, cfg)
    a = E.etc_layout_create(_model(order=0), _cfg(1))
    b = E.etc_layout_create(_model(order=1), _cfg(1))
    out = torch.zeros(4, dtype=torch.int64, device="cuda")
    with pytest.raises(E.EtcError) as e:                       # different row orders are different models
        E.etc_cost_matrix(a, b, out=(out, out, out))
    assert e.value.code == -3


@pytest.mark.parametrize("order", [0, 1])
def test_qkv_variants_scaled_c5(E, order):
    """s5 (config 5's GQA model scaled down: 16 q / 8 kv heads) from TP8 PP1 to TP16 PP1 (two ranks per KV group) and
    from TP16 back to TP4 PP2, both row orders."""
    w = workload("s5")
    m = dict(w["model"], qkv_order=order, vocab=4000 + 16 * 1)      # vocab divisible by 16
    for a, b in [(_cfg(8), _cfg(16)), (_cfg(16), _cfg(4, 2))]:
        for flags in (0, 1):
            g = _check_migration(E, m, a, b, w["seed"], flags=flags)
    assert g["plan"].stats.remote_bytes > 0
