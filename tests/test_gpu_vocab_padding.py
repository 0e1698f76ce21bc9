"""-m gpu parity of TP-dependent vocabulary padding (f3e, reading A31) through the whole CUDA path against the
element-wise oracle: padded cost matrices, traffic matrix, zero-fill descriptors (every destination byte is covered
exactly once by a slice or a fill), every destination buffer bit for bit — poisoned first, so a zero was written — in
one migration and in rounds of bounded staging."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload
from oracle import oracle as O
from helpers import make_logical, shard_all
from gpu_helpers import run_gpu_migration, upload, download
from test_vocab_padding_pins import CASES, _model, _cfg


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _check(E, model, old_cfg, new_cfg, seed, device_map=None, flags=0, payload="stamp"):
    oo, on = O.Layout(model, old_cfg), O.Layout(model, new_cfg)
    src = shard_all(oo, make_logical(model, seed, payload, lts=oo.logical_tensors()))
    g = run_gpu_migration(model, old_cfg, new_cfg, src, device_map=device_map, flags=flags)
    ov, need, hold = O.overlap(oo, on)
    assert np.array_equal(g["overlap"], ov) and np.array_equal(g["need"], need) and np.array_equal(g["hold"], hold)
    dm = g["device_map"]
    if device_map is None:
        ref = O.sketch_bruteforce(ov)[1] if ov.shape[1] <= 8 else O.sketch_hungarian(ov)[1]
        assert g["local_bytes"] == ref
    fill = np.zeros(on.n_dev, np.int64)
    dst, T, _ = O.migrate(oo, on, dm, src, fill_out=fill)
    st = g["plan"].stats
    assert np.array_equal(g["plan"].traffic(), T)
    local = int(np.trace(T)); remote = int(T.sum() - np.trace(T))
    assert st.local_bytes == local and st.remote_bytes == remote and st.fill_bytes == int(fill.sum())
    assert local + remote + st.fill_bytes == int(need.sum())
    for key, exp in dst.items():
        assert np.array_equal(g["dst"][key], exp), (key, int((g["dst"][key] != exp).sum()))
    # coverage: slices and fills together write every destination byte exactly once; fills per rank match the oracle
    cover = {key: np.zeros(v.shape[0] * v.itemsize, np.uint8) for key, v in dst.items()}
    fill_dev = np.zeros(on.n_dev, np.int64)
    recs = [(s, False) for which in (0, 1) for s in g["plan"].slices(which)] + [(s, True) for s in g["plan"].fills()]
    for s, is_fill in recs:
        key = (int(s["dst_rank"]), int(s["kind"]))
        for r in range(int(s["nrows"])):
            a = int(s["dst_off"]) + r * int(s["dst_stride"])
            cover[key][a:a + int(s["row_bytes"])] += 1
        if is_fill:
            assert int(s["src_dev"]) == -1 and int(s["dst_phys"]) == int(dm[key[0]])
            fill_dev[key[0]] += int(s["nrows"]) * int(s["row_bytes"])
    for key, c in cover.items():
        assert (c == 1).all(), key
    assert np.array_equal(fill_dev, fill)
    return g, int(fill.sum())


@pytest.mark.parametrize("i", range(len(CASES)))
def test_padded_vocab_tiny(E, i):
    m, a, b = CASES[i]
    rng = np.random.default_rng(70 + i)
    for flags in (0, 3):
        _check(E, m, a, b, 1700 + i, flags=flags)
    na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
    _check(E, m, a, b, 1750 + i, device_map=rng.permutation(max(na, nb))[:nb].astype(np.int32), payload="values")


def test_padded_vocab_scaled_gpt(E):
    """s2's model with the GPT-2 style odd vocabulary 3001 and divisor 16: TP2 PP2 DP2 (Vp 3008) -> TP4 PP2 DP1
    (Vp 3008... unit 64 -> 3008) and -> TP8 PP1 (unit 128 -> 3072, 64 rows zero-filled); tied embeddings."""
    w = workload("s2")
    m = dict(w["model"], vocab=3001, n_q_heads=8, n_kv_heads=8, head_dim=24)
    old = dict(w["old"], vocab_divisor=16)
    fills = []
    for new in (dict(w["new"], vocab_divisor=16), dict(tp=8, pp=1, dp=1, dist_opt=0, vocab_divisor=16),
                dict(tp=1, pp=2, dp=4, dist_opt=1, vocab_divisor=0 + 512)):
        for flags in (0, 1):
            g, f = _check(E, m, old, new, w["seed"], flags=flags)
        fills.append(f)
    assert fills[0] == 0 and fills[1] == 64 * 192 * 14 and fills[2] > 0


def test_padded_vocab_in_rounds(E):
    """kind-major rounds (f2): each kind's zero-fills go with its first round, while only that kind's buffers exist"""
    m, a, b = _model(vocab=11, tied=1), _cfg(1, 2, 2, 1, div=3), _cfg(4, 2, 1, 0, div=4)
    oo, on = O.Layout(m, a), O.Layout(m, b)
    src_np = shard_all(oo, make_logical(m, 5, "stamp", lts=oo.logical_tensors()))
    old, new = E.etc_layout_create(m, a), E.etc_layout_create(m, b)
    dm = np.arange(8, dtype=np.int32)[::-1].copy()
    plan = E.etc_plan_create(old, new, dm, E.ETC_KIND_MAJOR)
    assert plan.stats.fill_bytes > 0
    rounds = E.etc_plan_set_rounds(plan, 2 * 65536)
    staging = torch.empty(max(max(r.staging_bytes for r in rounds), 16), dtype=torch.uint8, device="cuda")
    out = {}
    for k in sorted(set(r.kind for r in rounds)):
        src_k = upload({key: v for key, v in src_np.items() if key[1] == k})
        dst_k = {key: v for key, v in E.alloc_buffers(new, fill=0x5A).items() if key[1] == k}
        for i, r in enumerate(rounds):
            if r.kind == k:
                E.etc_migrate_round(plan, i, src_k, dst_k, staging)
        torch.cuda.synchronize()
        for key, t in dst_k.items():
            out[key] = download(t, 4 if k else m["param_bytes"])
    dst, T, _ = O.migrate(oo, on, dm, src_np)
    for key, exp in dst.items():
        if exp.shape[0]:
            assert np.array_equal(out[key], exp), key


def test_padding_validation_codes_match_oracle(E):
    m = _model(vocab=5)
    for cfg in (_cfg(2, div=0), _cfg(2, div=-1)):
        with pytest.raises(O.OracleError) as oe:
            O.Layout(m, cfg)
        with pytest.raises(E.EtcError) as ge:
            E.etc_layout_create(m, cfg)
        assert ge.value.code == oe.value.code
    assert E.etc_layout_create(m, _cfg(2, div=1)).buffer_bytes(0, 1) == O.Layout(m, _cfg(2, div=1)).buffer_elems(0, 1) * 4


@pytest.mark.parametrize("seed", range(6))
def test_all_variants_combined_random_sweep(E, seed):
    """Every layout variant at once (helpers.random_variant_case): 10 random reconfigurations per seed through the whole
    CUDA path against the oracle, optimal and random device maps, LOCAL_DIRECT and ALL_STAGED | KIND_MAJOR."""
    from helpers import random_variant_case
    rng = np.random.default_rng(4000 + seed)
    filled = 0
    for i in range(10):
        m, a, b = random_variant_case(rng)
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        _, f = _check(E, m, a, b, 5000 + 100 * seed + i, flags=int(rng.choice([0, 1, 2, 3])))
        dm = rng.permutation(max(na, nb))[:nb].astype(np.int32)
        _, f2 = _check(E, m, a, b, 5050 + 100 * seed + i, device_map=dm, payload="values")
        filled += (f > 0) + (f2 > 0)
    print("cases with zero-fill:", filled)
