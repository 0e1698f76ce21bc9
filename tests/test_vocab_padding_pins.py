"""-m "not gpu": pins of the oracle's TP-dependent vocabulary padding (f3e, reading A31) against things other
than itself: hand-computed padded sizes (incl. the well-known 50257 -> 50304 / 50432 / 50688 / 51200 of Megatron-LM's
default divisor 128), hand-computed shard rows and zero-fill counts, and the P2-P10 battery restated for layouts whose
embedding tensors have different row counts: rows present on both sides are migrated (old padding rows included, so an
identity reconfiguration is the identity), rows beyond the old padded vocabulary are zero-filled, and the traffic
identity becomes  sum_o T[o][pi(n)] = need[n] - fill[n]."""
from __future__ import annotations
import numpy as np
import pytest

from etc_inputs.workloads import STYLE_GPT, STYLE_LLAMA
from etc_inputs import position_stamp
from oracle import oracle as O
from helpers import (read_golden, make_logical, shard_all, stamp_all, reassemble, resize_logical, replication_factor,
                     replication_map, random_variant_case)

GOLD = read_golden("vocab_padding_handcomputed.txt")


def _model(style=STYLE_GPT, vocab=5, tied=0, hidden=8, layers=2, kinds=0b1111, param_bytes=2):
    return dict(style=style, n_layers=layers, hidden=hidden, n_q_heads=8, n_kv_heads=8, head_dim=2, ffn_hidden=16,
                vocab=vocab, max_pos=4 if style == STYLE_GPT else 0, tied=tied, param_bytes=param_bytes, kinds=kinds)


def _cfg(tp, pp=1, dp=1, dist_opt=0, div=2):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt, vocab_divisor=div)


def _emb_ids(lts):
    """ids of the embedding tensors: word_embeddings (0) and lm_head (the last tensor, if it is vocab-shaped)"""
    ids = [0]
    if lts[-1][3] == 2 and lts[-1][2] == 1:          # post, COL  = lm_head (untied)
        ids.append(len(lts) - 1)
    return ids


@pytest.mark.parametrize("g", [g for g in GOLD if g[0] == "vp"], ids=lambda g: "-".join(g[1:4]))
def test_padded_rows_handcomputed(g):
    vocab, div, tp, want = int(g[1]), int(g[2]), int(g[3]), int(g[5])
    m = _model(vocab=vocab, hidden=8)
    lts = O.logical_tensors(m, _cfg(tp, div=div))
    assert lts[0][0] == want and lts[-1][0] == want            # word_embeddings and lm_head
    assert O.logical_tensors(m)[0][0] == vocab                 # the unpadded model
    L = O.Layout(m, _cfg(tp, div=div))
    assert sum(L.buffer_elems(r, 1) for r in range(tp)) - sum(
        O.Layout(dict(m, vocab=want), dict(tp=tp, pp=1, dp=1)).buffer_elems(r, 1) for r in range(tp)) == 0


@pytest.mark.parametrize("g", [g for g in GOLD if g[0] == "rows"], ids=lambda g: "-".join(g[1:3]))
def test_embedding_shard_rows_handcomputed(g):
    tp, r, want = int(g[1]), int(g[2]), [int(x) for x in g[4:]]
    for tied in (0, 1):
        m = _model(tied=tied)
        L = O.Layout(m, _cfg(tp))
        lt, _, row, col = L.global_of(r, 1)
        for t in _emb_ids(L.logical_tensors()):
            assert [int(x) for x in row[(lt == t) & (col == 0)]] == want


@pytest.mark.parametrize("g", [g for g in GOLD if g[0] == "fill"], ids=lambda g: "-".join(g[1:4]))
def test_zero_fill_counts_handcomputed(g):
    tp_o, tp_n, n, want = int(g[1]), int(g[2]), int(g[3]), int(g[5])
    for tied, n_emb in ((0, 2), (1, 1)):
        m = _model(tied=tied)
        old, new = O.Layout(m, _cfg(tp_o)), O.Layout(m, _cfg(tp_n))
        fill = np.zeros(new.n_dev, np.int64)
        dm = np.arange(new.n_dev, dtype=np.int32)
        O.migrate(old, new, dm, None, fill_out=fill)
        assert fill[n] == want * n_emb * (2 + 4 + 4 + 4)       # bf16 PARAM + fp32 MASTER, M, V


def check_padded_reconfiguration(model, old_cfg, new_cfg, seed, device_map=None):
    """The battery of tests/test_oracle_pins.py restated for layouts with different padded vocabularies."""
    old, new = O.Layout(model, old_cfg), O.Layout(model, new_cfg)
    lts_o, lts_n = old.logical_tensors(), new.logical_tensors()
    P = O.P_of(old, new)
    ov, need, hold = O.overlap(old, new)
    ov2, need2, hold2 = O.overlap(old, new, method="ranges")   # the separately written row-level routine agrees
    assert np.array_equal(ov, ov2) and np.array_equal(need, need2) and np.array_equal(hold, hold2)
    if device_map is None:
        device_map = O.sketch_bruteforce(ov)[0] if P <= 7 else O.sketch_hungarian(ov)[0]
    # --- P3: row sums with replication factors; an element beyond the other side's padded vocabulary is held 0 times
    def weighted(mine, dev, other, lts_other):
        tot = 0
        for k in mine.kinds():
            lt, _, row, col = mine.global_of(dev, k)
            for t in np.unique(lt):
                sel = (lt == t) & (row < lts_other[t][0])
                R = replication_map(other, k, lts_other, int(t))          # per element: KV-head replication varies it
                tot += int(R[row[sel], col[sel]].sum()) * O.kind_bytes(model, k)
        return tot
    for n in range(new.n_dev):
        assert ov[n].sum() == weighted(new, n, old, lts_o)
    for o in range(old.n_dev):
        assert ov[:, o].sum() == weighted(old, o, new, lts_n)
    # --- P8 / P4 with the index-stamped payload: new shards = shards of the resized logical tensors
    logical_o = make_logical(model, seed, "stamp", lts=lts_o)
    logical_n = resize_logical(logical_o, lts_n)
    src = shard_all(old, logical_o)
    fill = np.zeros(new.n_dev, np.int64)
    dst, T, _ = O.migrate(old, new, device_map, src, fill_out=fill)
    for n in range(new.n_dev):
        for k in new.kinds():
            assert np.array_equal(dst[(n, k)], new.shard_from_logical(n, k, logical_n[k])), ("P8", n, k)
    rebuilt, cover, consistent = reassemble(new, dst, logical_n)
    assert consistent
    for k in logical_n:
        for t in range(len(lts_n)):
            assert np.array_equal(rebuilt[k][t], logical_n[k][t]), ("P4", k, t)
            assert np.array_equal(cover[k][t], replication_map(new, k, lts_n, t))
    # --- fill: counted from global_of alone (elements of embedding tensors whose row lies beyond the old padded rows)
    for n in range(new.n_dev):
        want = 0
        for k in new.kinds():
            lt, _, row, _c = new.global_of(n, k)
            for t in _emb_ids(lts_n):
                want += int(((lt == t) & (row >= lts_o[t][0])).sum()) * O.kind_bytes(model, k)
        assert fill[n] == want
    # --- P3 on T: every needed byte has exactly one source, or is zero-filled
    for n in range(new.n_dev):
        assert T[:, device_map[n]].sum() == need[n] - fill[n]
    assert T.sum() == need.sum() - fill.sum()
    assert sum(int(T[device_map[n], device_map[n]]) for n in range(new.n_dev)) == sum(int(ov[n, device_map[n]]) for n in range(new.n_dev))
    # --- P9: position-stamped payload names the source; filled elements have none and are zero
    stamps = stamp_all(old)
    dst2, T2, _ = O.migrate(old, new, device_map, stamps)
    hist = np.zeros_like(T)
    for n in range(new.n_dev):
        for k in new.kinds():
            cnt = new.buffer_elems(n, k)
            if not cnt:
                continue
            sd, sl = O.source_of(old, new, device_map, n, k, np.arange(cnt))
            es = new.elem_bytes(k)
            assert (dst2[(n, k)][sd < 0] == 0).all()
            for o in np.unique(sd[sd >= 0]):
                sel = sd == o
                assert np.array_equal(dst2[(n, k)][sel], position_stamp(int(o), k, old.buffer_elems(int(o), k), es)[sl[sel]])
                hist[o, device_map[n]] += int(sel.sum()) * es
    assert np.array_equal(hist, T) and np.array_equal(T2, T)
    # --- P10 exactly once (filled elements are written once too)
    for n in range(new.n_dev):
        for k in new.kinds():
            cnt = new.buffer_elems(n, k)
            written = np.zeros(cnt, np.uint8)
            O.migrate_range(old, new, device_map, n, k, 0, cnt, None, None, None, written)
            assert (written == 1).all()
    return int(fill.sum())


CASES = [(_model(), _cfg(1), _cfg(2)), (_model(), _cfg(2), _cfg(1)), (_model(tied=1), _cfg(1, 2), _cfg(4, 2)),
         (_model(STYLE_LLAMA), _cfg(2, 1, 2, 1), _cfg(4, 1, 1)), (_model(STYLE_LLAMA, tied=1), _cfg(4, 2), _cfg(1, 2, 2, 1)),
         (_model(vocab=11), _cfg(1, 2, 2, 1, div=3), _cfg(2, 2, 2, 1, div=4)),          # dist-opt ranges cut the padding rows
         (_model(vocab=11, tied=1), _cfg(2, 2, 1, 0, div=4), _cfg(2, 1, 2, 0, div=0 + 1)),
         (_model(vocab=8), _cfg(2, 1, 1, 0, div=0), _cfg(4, 1, 1, 0, div=3)),          # unpadded -> padded
         (_model(vocab=8, tied=1), _cfg(4, 2, 1, 0, div=3), _cfg(2, 2, 1, 0, div=0))]  # padded -> unpadded


@pytest.mark.parametrize("i", range(len(CASES)))
def test_padded_vocab_full_battery(i):
    m, a, b = CASES[i]
    rng = np.random.default_rng(60 + i)
    check_padded_reconfiguration(m, a, b, 1600 + i)
    na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
    check_padded_reconfiguration(m, a, b, 1650 + i, device_map=rng.permutation(max(na, nb))[:nb].astype(np.int32))


def test_growth_fills_and_shrink_does_not():
    assert check_padded_reconfiguration(_model(), _cfg(1), _cfg(4), 3) > 0
    assert check_padded_reconfiguration(_model(), _cfg(4), _cfg(1), 4) == 0


def test_identity_reconfiguration_with_padding_is_the_identity():
    """P2: old padding rows are migrated like any other row, so old == new moves nothing and changes nothing."""
    for m, cfg in [(_model(), _cfg(2, 2, 2, 1)), (_model(STYLE_LLAMA, tied=1), _cfg(4, 2, 1, 0, div=3))]:
        old, new = O.Layout(m, cfg), O.Layout(m, cfg)
        ov, need, hold = O.overlap(old, new)
        assert np.array_equal(np.diag(ov), need) and np.array_equal(need, hold)
        src = shard_all(old, make_logical(m, 5, "values", lts=old.logical_tensors()))
        fill = np.zeros(new.n_dev, np.int64)
        dst, T, _ = O.migrate(old, new, np.arange(new.n_dev, dtype=np.int32), src, fill_out=fill)
        assert np.array_equal(T, np.diag(need)) and fill.sum() == 0
        for key in src:
            assert np.array_equal(src[key], dst[key])


def test_padding_validation():
    m = _model(vocab=5)
    with pytest.raises(O.OracleError) as e:                     # unpadded: vocab % tp (reading A12)
        O.Layout(m, _cfg(2, div=0))
    assert e.value.code == -2
    with pytest.raises(O.OracleError) as e:
        O.Layout(m, _cfg(2, div=-1))
    assert e.value.code == -1
    assert O.Layout(m, _cfg(2, div=1)).n_dev == 2               # divisor 1: pad to a multiple of tp only


@pytest.mark.parametrize("seed", range(4))
def test_all_variants_combined_random_sweep(seed):
    """Every layout variant at once (helpers.random_variant_case): the whole battery on 12 random reconfigurations per
    seed with optimal and random device maps."""
    rng = np.random.default_rng(3000 + seed)
    for i in range(12):
        m, a, b = random_variant_case(rng, max_devices=8)
        check_padded_reconfiguration(m, a, b, 2000 + 100 * seed + i)
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        check_padded_reconfiguration(m, a, b, 2050 + 100 * seed + i, device_map=rng.permutation(max(na, nb))[:nb].astype(np.int32))
