"""-m "not gpu": a second, differently built pin for the oracle's shard geometry.

`orc_global_of` computes (tensor, row, col) of a local element by index ARITHMETIC (block starts, divisions, moduli).  Here
the same shards are built the way Megatron-LM builds them — by ARRAY OPERATIONS on index tensors: `reshape` to
[kv_groups, q_per_group + 2, head_dim, hidden], `np.split` over the TP axis, `[gate; up]` chunking, `np.concatenate`
of the blocks, python list slicing for the pipeline split, flatten + pad + `reshape(dp, -1)` for the distributed
optimizer — and EVERY element of EVERY buffer is compared with the oracle (readings A9-A14, A27-A31).  A
misreading shared by the oracle and the CUDA layout builder (transposed split, wrong block order, off-by-one stage
boundary) cannot pass here unless it is also made in a third, structurally different construction.

The second test replaces the self-referential P9 block of test_oracle_pins.py: the source the oracle picks for an element
(`orc_source_of`, and through it `orc_migrate`) is re-derived in Python from `holders_of` alone, rule A6 written out."""
from __future__ import annotations
import numpy as np
import pytest

from etc_inputs import tiny_models, position_stamp
from etc_inputs.workloads import STYLE_GPT, STYLE_LLAMA
from oracle import oracle as O

REPL, COL, ROW, COL2, QKV = 0, 1, 2, 3, 4


def tensor_list(m, Vp):
    """[(name, rows, cols, split, where, layer)] in logical id order — DESIGN.md "Logical model", restated."""
    h, d, f = m["hidden"], m["head_dim"], m["ffn_hidden"]
    qkv, qd = (m["n_q_heads"] + 2 * m["n_kv_heads"]) * d, m["n_q_heads"] * d
    out = [("word_embeddings", Vp, h, COL, "pre", -1)]
    if m["style"] == STYLE_GPT and m["max_pos"] > 0:
        out.append(("position_embeddings", m["max_pos"], h, REPL, "pre", -1))
    for l in range(m["n_layers"]):
        if m["style"] == STYLE_GPT:
            out += [("ln1.w", 1, h, REPL, "layer", l), ("ln1.b", 1, h, REPL, "layer", l),
                    ("qkv.w", qkv, h, QKV, "layer", l), ("qkv.b", qkv, 1, QKV, "layer", l),
                    ("proj.w", h, qd, ROW, "layer", l), ("proj.b", 1, h, REPL, "layer", l),
                    ("ln2.w", 1, h, REPL, "layer", l), ("ln2.b", 1, h, REPL, "layer", l),
                    ("fc1.w", f, h, COL, "layer", l), ("fc1.b", f, 1, COL, "layer", l),
                    ("fc2.w", h, f, ROW, "layer", l), ("fc2.b", 1, h, REPL, "layer", l)]
        else:
            out += [("ln1.w", 1, h, REPL, "layer", l), ("qkv.w", qkv, h, QKV, "layer", l),
                    ("proj.w", h, qd, ROW, "layer", l), ("ln2.w", 1, h, REPL, "layer", l),
                    ("fc1.w", 2 * f, h, COL2, "layer", l), ("fc2.w", h, f, ROW, "layer", l)]
    out.append(("final_ln.w", 1, h, REPL, "post", -1))
    if m["style"] == STYLE_GPT:
        out.append(("final_ln.b", 1, h, REPL, "post", -1))
    if not m["tied"]:
        out.append(("lm_head", Vp, h, COL, "post", -1))
    return out


def tp_shard(m, idx, split, tp, r):
    """The TP shard of one logical tensor, given as a 2-D array `idx` of element ids, by array operations only."""
    if split == REPL:
        return idx
    if split == COL:
        return np.split(idx, tp, axis=0)[r]
    if split == ROW:
        return np.split(idx, tp, axis=1)[r]
    if split == COL2:                                   # SwiGLU fc1 = [gate; up]; a rank holds gate_r then up_r
        gate, up = np.split(idx, 2, axis=0)
        return np.concatenate([np.split(gate, tp, axis=0)[r], np.split(up, tp, axis=0)[r]], axis=0)
    q, k, d, cols = m["n_q_heads"], m["n_kv_heads"], m["head_dim"], idx.shape[1]
    qpg = q // k
    if m.get("qkv_order", 0) == 0:                      # Megatron's fused layout: [groups, q_per_group + 2, d, hidden]
        g4 = idx.reshape(k, qpg + 2, d, cols)
        if tp <= k:
            return np.split(g4, tp, axis=0)[r].reshape(-1, cols)
        rep = tp // k
        grp = g4[r // rep]                              # [qpg + 2, d, cols] of the rank's KV group
        q_share = np.split(grp[:qpg], rep, axis=0)[r % rep]
        return np.concatenate([q_share.reshape(-1, cols), grp[qpg:].reshape(-1, cols)], axis=0)
    Q, K, V = idx[: q * d].reshape(q, d, cols), idx[q * d:(q + k) * d].reshape(k, d, cols), idx[(q + k) * d:].reshape(k, d, cols)
    if tp <= k:
        parts = [np.split(Q, tp, axis=0)[r], np.split(K, tp, axis=0)[r], np.split(V, tp, axis=0)[r]]
    else:
        g = r // (tp // k)
        parts = [np.split(Q, tp, axis=0)[r], K[g:g + 1], V[g:g + 1]]
    return np.concatenate([p.reshape(-1, cols) for p in parts], axis=0)


def stage_layers(n_layers, c):
    layers = list(range(n_layers))
    first, last, pp = c.get("pp_first", 0), c.get("pp_last", 0), c["pp"]
    if not first and not last:
        return [list(x) for x in np.split(np.array(layers), pp)]
    head = [layers[:first]] if first else []
    tail = [layers[n_layers - last:]] if last else []
    mid = layers[first:n_layers - last if last else n_layers]
    n_mid = pp - len(head) - len(tail)
    mids = [list(x) for x in np.split(np.array(mid), n_mid)] if n_mid else []
    return head + mids + tail


def build_buffers(m, c):
    """{(dev, kind): (tensor id array, flat logical index array, post-copy flag array)} by array operations."""
    tp, pp, dp = c["tp"], c["pp"], c["dp"]
    div = c.get("vocab_divisor", 0)
    Vp = m["vocab"] if div <= 0 else -(-m["vocab"] // (div * tp)) * div * tp
    tl = tensor_list(m, Vp)
    per_stage = stage_layers(m["n_layers"], c)
    out = {}
    for s in range(pp):
        for r in range(tp):
            tid, flat, post = [], [], []

            def add(t, replica=False):
                name, rows, cols, split, where, layer = tl[t]
                ids = np.arange(rows * cols, dtype=np.int64).reshape(rows, cols)
                sh = tp_shard(m, ids, split, tp, r).ravel()
                tid.append(np.full(sh.shape[0], t, np.int32)); flat.append(sh)
                post.append(np.full(sh.shape[0], 1 if replica else 0, np.int32))
            for t, x in enumerate(tl):
                if x[4] == "pre" and s == 0:
                    add(t)
            for t, x in enumerate(tl):
                if x[4] == "layer" and x[5] in per_stage[s]:
                    add(t)
            for t, x in enumerate(tl):
                if x[4] == "post" and s == pp - 1:
                    add(t)
            if m["tied"] and pp > 1 and s == pp - 1:
                add(0, replica=True)                    # the output layer's copy of word_embeddings (reading A11)
            tid, flat, post = np.concatenate(tid), np.concatenate(flat), np.concatenate(post)
            for d in range(dp):
                dev = r + tp * (d + dp * s)
                for k in range(4):
                    if not (m["kinds"] >> k) & 1:
                        continue
                    if c.get("dist_opt", 0) and dp > 1 and k >= 1:
                        a = max(1, c.get("dist_opt_align", 0))
                        n = tid.shape[0]
                        padded = -(-n // (dp * a)) * dp * a          # Megatron pads the flat buffer, then views it [dp, -1]
                        sel = np.arange(padded).reshape(dp, -1)[d]
                        sel = sel[sel < n]
                        out[(dev, k)] = (tid[sel], flat[sel], post[sel])
                    else:
                        out[(dev, k)] = (tid, flat, post)
    return tl, out


def _model(style=STYLE_LLAMA, order=0, n_q=4, n_kv=2, d=2, layers=4, hidden=8, tied=0, kinds=0b1111, vocab=16, ffn=16,
           pbytes=2):
    return dict(style=style, n_layers=layers, hidden=hidden, n_q_heads=n_q, n_kv_heads=n_kv, head_dim=d, ffn_hidden=ffn,
                vocab=vocab, max_pos=4 if style == STYLE_GPT else 0, tied=tied, param_bytes=pbytes, kinds=kinds,
                qkv_order=order)


def _cfg(tp, pp=1, dp=1, dist_opt=0, **kw):
    return dict(dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt, pp_first=0, pp_last=0, dist_opt_align=0, vocab_divisor=0), **kw)


CASES = [
    (_model(STYLE_GPT, 0, n_q=4, n_kv=4, tied=1), _cfg(2, 2, 2, 1)),                       # MHA, tied, dist-opt
    (_model(STYLE_GPT, 0, n_q=4, n_kv=4, tied=0, hidden=12, d=3), _cfg(4, 1, 3, 1)),       # dist-opt range cuts rows
    (_model(STYLE_LLAMA, 0, n_q=8, n_kv=2, hidden=16), _cfg(2, 2, 1)),                     # GQA groups + SwiGLU COL2
    (_model(STYLE_LLAMA, 1, n_q=8, n_kv=2, hidden=16), _cfg(2, 2, 1)),                     # [Q;K;V] order
    (_model(STYLE_LLAMA, 0, n_q=8, n_kv=2, hidden=16), _cfg(8, 1, 2, 1)),                  # KV-head replication, grouped
    (_model(STYLE_LLAMA, 1, n_q=8, n_kv=2, hidden=16), _cfg(4, 2, 2, 1)),                  # KV-head replication, [Q;K;V]
    (_model(STYLE_GPT, 1, n_q=8, n_kv=4, hidden=16, tied=1, layers=6), _cfg(8, 3, 1)),     # replication + tied + bias
    (_model(STYLE_GPT, 0, layers=7, tied=1, n_q=4, n_kv=4), _cfg(2, 3, 1, 0, pp_first=1)),  # uneven: 1 + 3 + 3
    (_model(STYLE_LLAMA, 0, layers=8), _cfg(1, 4, 2, 1, pp_first=1, pp_last=3)),           # uneven: 1 + 2 + 2 + 3
    (_model(STYLE_GPT, 0, n_q=4, n_kv=4, vocab=13, tied=1), _cfg(2, 2, 1, 0, vocab_divisor=4)),   # padded vocabulary
    (_model(STYLE_LLAMA, 0, vocab=11), _cfg(4, 1, 2, 1, vocab_divisor=3, dist_opt_align=8)),      # padding + aligned dist-opt
    (_model(STYLE_LLAMA, 0, n_q=4, n_kv=4, kinds=0b0110, pbytes=4), _cfg(2, 2, 3, 1, dist_opt_align=24)),
]
CASES += [(m, _cfg(tp, pp, dp, do)) for _, m in tiny_models()
          for tp, pp, dp, do in ((1, 1, 1, 0), (2, 2, 1, 0), (2, 1, 2, 1), (1, 2, 4, 1))]


@pytest.mark.parametrize("i", range(len(CASES)))
def test_every_element_matches_the_array_construction(i):
    m, c = CASES[i]
    try:
        lay = O.Layout(m, c)
    except O.OracleError:
        pytest.skip("configuration not valid for this model")
    tl, bufs = build_buffers(m, c)
    o_tl = lay.logical_tensors()
    assert [(x[1], x[2], x[3]) for x in tl] == [(x[0], x[1], x[2]) for x in o_tl]          # shapes and split types
    assert lay.n_dev == c["tp"] * c["pp"] * c["dp"]
    n_checked = 0
    for dev in range(lay.n_dev):
        for k in range(4):
            cnt = lay.buffer_elems(dev, k)
            if not (m["kinds"] >> k) & 1:
                assert cnt == 0
                continue
            tid, flat, post = bufs[(dev, k)]
            assert cnt == tid.shape[0], (dev, k)
            if cnt == 0:
                continue
            lt, pc, row, col = lay.global_of(dev, k)
            cols = np.array([x[2] for x in tl], np.int64)[lt]
            assert np.array_equal(lt, tid), (dev, k)
            assert np.array_equal(row * cols + col, flat), (dev, k)
            assert np.array_equal(pc, post), (dev, k)
            n_checked += cnt
    assert n_checked > 0


def _coords(c, dev):
    return (dev // c["tp"]) % c["dp"], dev // (c["tp"] * c["dp"]), dev % c["tp"]            # d, s, r


SRC_CASES = [
    (_model(STYLE_GPT, 0, n_q=4, n_kv=4, tied=1), _cfg(2, 2, 2, 0), _cfg(1, 2, 4, 0)),       # DP growth round-robin, tied
    (_model(STYLE_GPT, 0, n_q=4, n_kv=4, tied=1), _cfg(2, 2, 2, 1), _cfg(4, 1, 2, 1)),       # dist-opt both sides
    (_model(STYLE_LLAMA, 0, n_q=8, n_kv=2, hidden=16), _cfg(8, 1, 1), _cfg(2, 2, 2)),        # replicated K/V heads as sources
    (_model(STYLE_LLAMA, 1, n_q=8, n_kv=2, hidden=16), _cfg(4, 1, 2, 1), _cfg(8, 1, 1)),
    (_model(STYLE_GPT, 0, layers=6, n_q=4, n_kv=4), _cfg(2, 3, 1), _cfg(2, 2, 2)),           # scale-out onto fresh devices
]


@pytest.mark.parametrize("i", range(len(SRC_CASES)))
def test_sources_rederived_from_holders(i):
    """Reading A6 written out over `holders_of` (no failures): (i) the destination's own physical device if it holds the
    element; (ii) else stage = the holding stage (first stage for the pre copy, last stage for the post copy of the tied
    embedding), TP rank = ranks[r' mod count] over the ascending TP ranks of that stage holding it, DP rank = the one
    holding it if the kind is DP-sharded, else d' mod dp_old.  Compared with orc_source_of AND, through a position-
    stamped payload, with what orc_migrate actually copied."""
    m, a, b = SRC_CASES[i]
    oo, on = O.Layout(m, a), O.Layout(m, b)
    rng = np.random.default_rng(40 + i)
    P = max(oo.n_dev, on.n_dev)
    for trial in range(2):
        dm = (np.arange(on.n_dev) if trial == 0 else rng.permutation(P)[: on.n_dev]).astype(np.int32)
        stamps = {(d, k): position_stamp(d, k, oo.buffer_elems(d, k), oo.elem_bytes(k)) for d in range(oo.n_dev) for k in oo.kinds()}
        dst, T, _ = O.migrate(oo, on, dm, stamps)
        hist = np.zeros_like(T)
        for n in range(on.n_dev):
            d_new, s_new, r_new = _coords(b, n)
            p = int(dm[n])
            for k in on.kinds():
                cnt = on.buffer_elems(n, k)
                if not cnt:
                    continue
                sd, sl = O.source_of(oo, on, dm, n, k, np.arange(cnt))
                lt, pc, row, col = on.global_of(n, k)
                es = on.elem_bytes(k)
                dp_sharded = a["dist_opt"] and a["dp"] > 1 and k >= 1
                for e in range(cnt):
                    holders = oo.holders_of(k, int(lt[e]), int(row[e]), int(col[e]))
                    mine = [h for h in holders if h[0] == p]
                    if mine:
                        want = mine[0]
                    else:
                        stages = sorted({_coords(a, dev)[1] for dev, _ in holders})
                        s_des = stages[-1] if (pc[e] and len(stages) > 1) else stages[0]
                        on_stage = [h for h in holders if _coords(a, h[0])[1] == s_des]
                        ranks = sorted({_coords(a, dev)[2] for dev, _ in on_stage})
                        r_des = ranks[r_new % len(ranks)]
                        cands = [h for h in on_stage if _coords(a, h[0])[2] == r_des]
                        if dp_sharded:
                            assert len(cands) == 1
                            want = cands[0]
                        else:
                            want = next(h for h in cands if _coords(a, h[0])[0] == d_new % a["dp"])
                    assert (int(sd[e]), int(sl[e])) == want, (n, k, e)
                    assert dst[(n, k)][e] == stamps[(want[0], k)][want[1]], (n, k, e)
                    hist[want[0], p] += es
        assert np.array_equal(hist, T)
