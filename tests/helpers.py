"""Test helpers that use ONLY the oracle and the seeded input generators (never the CUDA path)."""
from __future__ import annotations
import os
import numpy as np
from etc_inputs import logical_values, index_stamp, position_stamp
from oracle import oracle as O

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


def make_logical(model: dict, seed: int, payload: str = "values", lts=None):
    """{kind: [2-D array per logical tensor]} in logical space (uint16 / uint32 bit patterns).  lts: the tensor list to
    use instead of the unpadded model's (a layout's own list when the vocabulary is padded, reading A31)."""
    lts = O.logical_tensors(model) if lts is None else lts
    out = {}
    for k in range(4):
        if not (model["kinds"] >> k) & 1:
            continue
        es = O.kind_bytes(model, k)
        arrs = []
        for t, (rows, cols, *_r) in enumerate(lts):
            n = rows * cols
            if payload == "values":
                v = logical_values(seed, k, t, n, es)
            elif payload == "salted":                      # index stamp that also depends on the seed (cheap to make)
                v = index_stamp(k, t, n, es, salt=seed)
            else:
                v = index_stamp(k, t, n, es)
            arrs.append(v.reshape(rows, cols))
        out[k] = arrs
    return out


def shard_all(layout: O.Layout, logical: dict):
    """{(dev, kind): 1-D array} — the oracle cuts every buffer out of the logical tensors."""
    return {(d, k): layout.shard_from_logical(d, k, logical[k]) for d in range(layout.n_dev) for k in layout.kinds()}


# ---- memoised oracle results.  Many -m gpu tests run the SAME reconfiguration (same layouts, same payload, same device
# map) through different launch modes of the CUDA path; the oracle's answer does not depend on the mode, so it is
# computed once per distinct input and reused (it is the slowest part of those tests by far).
import collections
import json

_MEMO: "collections.OrderedDict" = collections.OrderedDict()


def _memo(key, fn, keep=16):
    if key in _MEMO:
        _MEMO.move_to_end(key)
        return _MEMO[key]
    val = fn()
    _MEMO[key] = val
    while len(_MEMO) > keep:
        _MEMO.popitem(last=False)
    return val


def _lkey(layout: O.Layout):
    failed = getattr(layout, "failed", None)
    return (json.dumps(layout.model, sort_keys=True), json.dumps(layout.cfg, sort_keys=True),
            None if failed is None else bytes(failed))


class KeyedBufs(dict):
    """{(dev, kind): array} that remembers what it was made from (see oracle_migrate).  Treat as read-only."""
    key = None


def sharded_payload(layout: O.Layout, seed: int, payload: str = "stamp", padded_lts: bool = False) -> KeyedBufs:
    """shard_all(layout, make_logical(layout.model, seed, payload)), memoised."""
    key = ("shards", _lkey(layout)[:2], int(seed), payload, bool(padded_lts))

    def make():
        lts = layout.logical_tensors() if padded_lts else None
        out = KeyedBufs(shard_all(layout, make_logical(layout.model, seed, payload, lts=lts)))
        out.key = key
        return out
    return _memo(key, make)


def oracle_overlap(old: O.Layout, new: O.Layout, method: str = "elementwise"):
    """O.overlap(old, new, method=...) -> (overlap, need, hold), memoised (no failure masks)."""
    if getattr(old, "failed", None) is not None:
        return O.overlap(old, new, method=method)
    return _memo(("overlap", _lkey(old), _lkey(new), method), lambda: O.overlap(old, new, method=method))


def oracle_migrate(old: O.Layout, new: O.Layout, device_map, src_bufs):
    """O.migrate(old, new, device_map, src_bufs) -> (dst, T, overrides); memoised when src_bufs came from
    sharded_payload (its key names the payload)."""
    dm = np.ascontiguousarray(device_map, np.int32)
    skey = getattr(src_bufs, "key", None)
    if skey is None:
        return O.migrate(old, new, dm, src_bufs)
    return _memo(("migrate", _lkey(old), _lkey(new), dm.tobytes(), skey), lambda: O.migrate(old, new, dm, src_bufs))


def stamp_all(layout: O.Layout):
    """{(dev, kind): position-stamped 1-D array} (pin P9: values name the buffer and position they came from)."""
    return {(d, k): position_stamp(d, k, layout.buffer_elems(d, k), layout.elem_bytes(k))
            for d in range(layout.n_dev) for k in layout.kinds()}


def reassemble(layout: O.Layout, bufs: dict, logical_like: dict):
    """Rebuild every logical tensor from shard buffers.  Returns (rebuilt {kind: [arrays]}, cover {kind: [counts]},
    consistent: bool) — cover counts how many buffers held each element; consistent is False if replicas differ."""
    rebuilt = {k: [np.zeros_like(a) for a in v] for k, v in logical_like.items()}
    cover = {k: [np.zeros(a.shape, np.int32) for a in v] for k, v in logical_like.items()}
    consistent = True
    for (d, k), buf in bufs.items():
        if buf.shape[0] == 0:
            continue
        lt, _, row, col = layout.global_of(d, k)
        for t in np.unique(lt):
            sel = lt == t
            r, c = row[sel], col[sel]
            seen = cover[k][t][r, c] > 0
            if seen.any() and not np.array_equal(rebuilt[k][t][r[seen], c[seen]], buf[sel][seen]):
                consistent = False
            rebuilt[k][t][r, c] = buf[sel]
            np.add.at(cover[k][t], (r, c), 1)
    return rebuilt, cover, consistent


def replication_factor(layout: O.Layout, kind: int, split: int, t: int) -> int:
    """R(t) of pin P3: how many buffers hold each element of tensor t of this kind."""
    c, m = layout.cfg, layout.model
    f = c["tp"] if split == 0 else 1
    dp_sharded = c.get("dist_opt", 0) and c["dp"] > 1 and kind >= 1
    f *= 1 if dp_sharded else c["dp"]
    if m["tied"] and c["pp"] > 1 and t == 0:
        f *= 2
    return f


def replication_map(layout: O.Layout, kind: int, lt_info, t: int) -> np.ndarray:
    """R(t) of pin P3 per ELEMENT: how many buffers of `kind` hold each element of logical tensor t, written from the
    definitions (readings A6, A10, A11, A14, A29, A30), not from the oracle: replicated tensors are on every TP
    rank, a kind that is not DP-sharded is on every DP rank, the tied embedding is on two stages, and under KV-head
    replication (tp > n_kv) the rows of a K or V head are on tp/n_kv TP ranks."""
    rows, cols, split = lt_info[t][0], lt_info[t][1], lt_info[t][2]
    c, m = layout.cfg, layout.model
    R = np.full((rows, cols), replication_factor(layout, kind, split, t), np.int64)
    if split == 4 and c["tp"] > m["n_kv_heads"]:                 # fused QKV (weight or bias) with replicated KV heads
        rep = c["tp"] // m["n_kv_heads"]
        d, q, k = m["head_dim"], m["n_q_heads"], m["n_kv_heads"]
        r = np.arange(rows)
        if m.get("qkv_order", 0) == 0:
            is_kv = (r % ((q // k + 2) * d)) >= (q // k) * d     # inside a group: q heads first, then K, then V
        else:
            is_kv = r >= q * d                                   # [Q; K; V]
        R[is_kv, :] *= rep
    return R


def resize_logical(logical: dict, lts_to) -> dict:
    """Reading A31 stated on logical tensors: going to a layout whose embedding tensors have another padded row count,
    rows present on both sides are kept, rows beyond the new count are dropped, rows beyond the old count are zero."""
    out = {}
    for k, arrs in logical.items():
        new = []
        for a, (rows, cols, *_r) in zip(arrs, lts_to):
            assert a.shape[1] == cols
            b = np.zeros((rows, cols), a.dtype)
            m = min(rows, a.shape[0])
            b[:m] = a[:m]
            new.append(b)
        out[k] = new
    return out


def random_variant_case(rng, max_devices=12):
    """A random tiny (model, old cfg, new cfg) drawing on EVERY layout variant at once (both styles, GQA ratios, both QKV
    row orders, KV-head replication, tied / untied, uneven pipeline splits, distributed optimizer with and without
    alignment, padded and unpadded vocabularies, any subset of state kinds), both configurations valid for the oracle."""
    while True:
        n_kv = int(rng.choice([1, 2, 4])); qpg = int(rng.choice([1, 2, 4]))
        style = int(rng.integers(0, 2))
        model = dict(style=style, n_layers=int(rng.choice([2, 3, 4, 6])), hidden=int(rng.choice([8, 12])),
                     n_q_heads=n_kv * qpg, n_kv_heads=n_kv, head_dim=int(rng.choice([2, 3])),
                     ffn_hidden=int(rng.choice([16, 24])), vocab=int(rng.choice([8, 11, 13, 16])),
                     max_pos=int(rng.choice([0, 5])) if style == 0 else 0, tied=int(rng.integers(0, 2)),
                     param_bytes=int(rng.choice([2, 4])), kinds=int(rng.integers(1, 16)), qkv_order=int(rng.integers(0, 2)))
        cfgs = []
        for _ in range(2):
            pp = int(rng.choice([1, 2, 3]))
            c = dict(tp=int(rng.choice([1, 2, 4, 8])), pp=pp, dp=int(rng.choice([1, 2, 3])), dist_opt=int(rng.integers(0, 2)),
                     pp_first=0, pp_last=0, dist_opt_align=int(rng.choice([0, 0, 8, 24])),
                     vocab_divisor=int(rng.choice([0, 0, 1, 3, 4])))
            if pp >= 2 and rng.integers(0, 3) == 0:
                c["pp_first"] = int(rng.integers(1, 3))
            if pp >= 2 and rng.integers(0, 4) == 0:
                c["pp_last"] = int(rng.integers(1, 3))
            cfgs.append(c)
        if any(c["tp"] * c["pp"] * c["dp"] > max_devices for c in cfgs):
            continue
        try:
            O.Layout(model, cfgs[0]); O.Layout(model, cfgs[1])
        except O.OracleError:
            continue
        return model, cfgs[0], cfgs[1]
