"""-m "not gpu": pins of the oracle's fused-QKV layout variants (f3): [Q;K;V] block order (reading A29) and KV-head
replication when tp > n_kv (reading A30), against hand-computed shard contents, the attention-consistency property (a
rank must hold the K and V head of every q head it holds, and nothing else), and the P2-P10 battery."""
from __future__ import annotations
import numpy as np
import pytest

from etc_inputs.workloads import STYLE_GPT, STYLE_LLAMA
from oracle import oracle as O
from helpers import read_golden
from test_oracle_pins import _check_reconfiguration

GOLD = read_golden("qkv_variants_handcomputed.txt")


def _model(style=STYLE_LLAMA, order=0, n_q=4, n_kv=2, d=2, layers=2, hidden=8, tied=0, kinds=0b1111):
    return dict(style=style, n_layers=layers, hidden=hidden, n_q_heads=n_q, n_kv_heads=n_kv, head_dim=d, ffn_hidden=16,
                vocab=8, max_pos=4 if style == STYLE_GPT else 0, tied=tied, param_bytes=2, kinds=kinds, qkv_order=order)


def _cfg(tp, pp=1, dp=1, dist_opt=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt)


def _qkv_rows(L, model, dev, kind=0, layer=0, weight=True):
    """logical rows of the QKV weight (or bias) of `layer` held by `dev`, in local order (one entry per row)."""
    lts = O.logical_tensors(model)
    ids = [i for i, t in enumerate(lts) if t[2] == 4 and t[4] == layer]
    t = ids[0] if weight else ids[1]
    lt, _, row, col = L.global_of(dev, kind)
    sel = (lt == t) & (col == 0)
    return [int(x) for x in row[sel]]


@pytest.mark.parametrize("g", GOLD, ids=lambda r: "-".join(r[1:4]))
def test_qkv_shard_rows_handcomputed(g):
    order, tp, r = int(g[1]), int(g[2]), int(g[3])
    want = [int(x) for x in g[5:]]
    for style in (STYLE_LLAMA, STYLE_GPT):
        model = _model(style, order)
        L = O.Layout(model, _cfg(tp))
        assert _qkv_rows(L, model, r) == want
        if style == STYLE_GPT:
            assert _qkv_rows(L, model, r, weight=False) == want          # the bias is split like the weight
        assert _qkv_rows(L, model, r, kind=2, layer=1) == want           # every layer, every kind


def _heads(model, rows):
    """(set of q heads, set of k heads, set of v heads) a list of logical QKV rows covers, from the definition of the
    two row orders; every head must be covered completely."""
    q, k, d = model["n_q_heads"], model["n_kv_heads"], model["head_dim"]
    qpg = q // k
    out = (set(), set(), set())
    count = {}
    for r in rows:
        if model["qkv_order"] == 0:
            g, w = divmod(r, (qpg + 2) * d)
            h = w // d
            key = (0, g * qpg + h) if h < qpg else ((1, g) if h == qpg else (2, g))
        else:
            key = (0, r // d) if r < q * d else ((1, (r - q * d) // d) if r < (q + k) * d else (2, (r - (q + k) * d) // d))
        count[key] = count.get(key, 0) + 1
    for (typ, h), c in count.items():
        assert c == d, "a head is cut"
        out[typ].add(h)
    return out


@pytest.mark.parametrize("order", [0, 1])
@pytest.mark.parametrize("n_q,n_kv,tp", [(8, 8, 4), (8, 2, 2), (8, 2, 4), (8, 2, 8), (12, 3, 6), (16, 4, 16), (4, 1, 4), (6, 1, 2)])
def test_attention_consistency(order, n_q, n_kv, tp):
    """GQA-aware split: every rank holds n_q/tp whole q heads, exactly the K and V heads of their groups, all ranks
    together hold every q head once and every K/V head max(1, tp/n_kv) times."""
    model = dict(_model(order=order, n_q=n_q, n_kv=n_kv, d=2, hidden=n_q * 2), ffn_hidden=48, vocab=48)
    L = O.Layout(model, _cfg(tp))
    qpg = n_q // n_kv
    seen_q, seen_kv = [], []
    for r in range(tp):
        qs, ks, vs = _heads(model, _qkv_rows(L, model, r))
        assert len(qs) == n_q // tp
        assert ks == vs == {h // qpg for h in qs}
        seen_q += sorted(qs); seen_kv += sorted(ks)
    assert sorted(seen_q) == list(range(n_q))
    rep = max(1, tp // n_kv)
    assert sorted(seen_kv) == sorted(list(range(n_kv)) * rep)


def test_invalid_qkv_variants():
    for model, cfg, code in [(_model(n_q=8, n_kv=4, hidden=24), _cfg(3), -2),  # tp <= n_kv: n_kv % tp
                             (_model(n_q=8, n_kv=2), _cfg(6), -6),            # tp % n_kv
                             (_model(n_q=6, n_kv=2, hidden=12), _cfg(4), -6), # q heads of a group do not split over 2 ranks
                             (_model(order=2), _cfg(1), -1)]:
        with pytest.raises(O.OracleError) as e:
            O.Layout(model, cfg)
        assert e.value.code == code, (model, cfg)


def test_order_relabelling_does_not_change_group_order_bits():
    """Reading A10's note: with tp <= n_kv the two row orders are relabellings of each other, so every cost matrix is
    identical; the shard BYTES differ only by the row permutation."""
    for tp_old, tp_new in [(1, 2), (2, 1), (2, 2)]:
        ovs = []
        for order in (0, 1):
            m = _model(order=order)
            ov, need, hold = O.overlap(O.Layout(m, _cfg(tp_old, 2)), O.Layout(m, _cfg(tp_new, 1, 2)))
            ovs.append((ov, need, hold))
        for a, b in zip(*ovs):
            assert np.array_equal(a, b)


def test_qkv_variants_full_battery():
    """P2-P5, P8-P10 on reconfigurations into, out of and between KV-replicated layouts, both row orders, both styles,
    with PP / DP / dist-opt changes and arbitrary device maps."""
    cases = [(_model(STYLE_LLAMA, 0), _cfg(2), _cfg(4)), (_model(STYLE_LLAMA, 0), _cfg(4), _cfg(1, 2)),
             (_model(STYLE_LLAMA, 1), _cfg(1, 2), _cfg(2)), (_model(STYLE_LLAMA, 1), _cfg(4), _cfg(2, 1, 2)),
             (_model(STYLE_GPT, 1, tied=1), _cfg(4, 2), _cfg(2, 1, 2, 1)), (_model(STYLE_GPT, 0, tied=1), _cfg(2, 1, 2, 1), _cfg(4, 2)),
             (_model(STYLE_LLAMA, 0, n_q=8, n_kv=2, hidden=16), _cfg(8), _cfg(4, 1, 2, 1)),
             (_model(STYLE_LLAMA, 1, n_q=8, n_kv=2, hidden=16), _cfg(4, 1, 2, 1), _cfg(8)),
             (_model(STYLE_LLAMA, 0, n_q=4, n_kv=1), _cfg(4), _cfg(2, 2))]
    rng = np.random.default_rng(17)
    for i, (m, a, b) in enumerate(cases):
        assert _check_reconfiguration(m, a, b, 1400 + i)
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        dm = rng.permutation(max(na, nb))[:nb].astype(np.int32)
        assert _check_reconfiguration(m, a, b, 1450 + i, device_map=dm)
