"""Pins for the CPU oracle: the oracle is checked against what the paper and the
mathematics fix — never against itself and never against the CUDA path."""
from __future__ import annotations
import itertools
import numpy as np
import pytest

from etc_inputs import workload, tiny_models, tiny_parallel_cfgs, position_stamp, STYLE_GPT
from oracle import oracle as O
from helpers import read_golden, make_logical, shard_all, stamp_all, reassemble, replication_factor, replication_map

TINY = dict(tiny_models())


def _layouts(model, old, new):
    try:
        return O.Layout(model, old), O.Layout(model, new)
    except O.OracleError:
        return None, None


# ------------------------------------------------------------------ layout: hand-computed global_of (golden)
def test_layout_handcomputed_golden():
    """global_of against values derived by hand from the tensor table and layout rules (tests/golden)."""
    cache = {}
    for row in read_golden("layout_handcomputed.txt"):
        name, tp, pp, dp, do, dev, kind = row[0], *map(int, row[1:7])
        key = (name, tp, pp, dp, do)
        if key not in cache:
            cache[key] = O.Layout(TINY[name], dict(tp=tp, pp=pp, dp=dp, dist_opt=do))
        L = cache[key]
        if row[7] == "count":
            assert L.buffer_elems(dev, kind) == int(row[8]), row
            continue
        l = int(row[7])
        lt, pc, r, c = L.global_of(dev, kind, l, 1)
        assert [int(lt[0]), int(pc[0]), int(r[0]), int(c[0])] == list(map(int, row[8:12])), row


def test_holders_of_is_inverse_of_global_of():
    """holders_of (arithmetic) == brute-force inversion of global_of over every device and local index."""
    for name, model in tiny_models():
        for cfg in (dict(tp=2, pp=2, dp=2, dist_opt=1), dict(tp=2, pp=1, dp=2, dist_opt=0),
                    dict(tp=1, pp=2, dp=3, dist_opt=1)):
            try:
                L = O.Layout(model, cfg)
            except O.OracleError:
                continue
            for k in L.kinds():
                inv = {}
                for d in range(L.n_dev):
                    lt, pc, row, col = L.global_of(d, k)
                    for l in range(lt.shape[0]):
                        inv.setdefault((int(lt[l]), int(row[l]), int(col[l])), []).append((d, l))
                lts = O.logical_tensors(model)
                # every logical element is held somewhere, and holders_of lists exactly the brute-force holders
                keys = list(inv.keys())
                assert len(keys) == sum(r * c for r, c, *_ in lts)
                step = max(1, len(keys) // 400)
                for key in keys[::step]:
                    assert sorted(L.holders_of(k, *key)) == sorted(inv[key]), (name, cfg, k, key)


def test_every_device_holds_distinct_elements():
    for name, model in tiny_models():
        L = O.Layout(model, dict(tp=2, pp=2, dp=2, dist_opt=1))
        for d in range(L.n_dev):
            for k in L.kinds():
                lt, pc, row, col = L.global_of(d, k)
                keys = set(zip(lt.tolist(), row.tolist(), col.tolist()))
                assert len(keys) == lt.shape[0]


def test_validation_errors():
    m = dict(TINY["gpt_np"])
    with pytest.raises(O.OracleError) as e:
        O.Layout(m, dict(tp=1, pp=3, dp=1, dist_opt=0))       # 4 layers % 3
    assert e.value.code == -2
    with pytest.raises(O.OracleError) as e:
        O.Layout(m, dict(tp=4, pp=1, dp=1, dist_opt=0))       # tp > kv heads (A10)
    assert e.value.code == -6


# ------------------------------------------------------------------ P1: the paper's worked example
def test_P1_paper_fig4_pp4_to_pp2():
    """16 layers, PP4 -> PP2: c_{0,0} = 4 (layer units), full matrix by c = len(curr)-len(curr∩prev)."""
    gold = np.array([[int(x) for x in r] for r in read_golden("paper_fig4_pp4_to_pp2.txt")])
    model = dict(style=STYLE_GPT, n_layers=16, hidden=8, n_q_heads=2, n_kv_heads=2, head_dim=4, ffn_hidden=16,
                 vocab=8, max_pos=4, tied=0, param_bytes=2, kinds=0b1111)
    old, new = O.Layout(model, dict(tp=1, pp=4, dp=1, dist_opt=0)), O.Layout(model, dict(tp=1, pp=2, dp=1, dist_opt=0))
    ov, need, hold = O.overlap(old, new, only_layers=True)
    per_layer = hold[0] // 4                      # prev rank 0 holds 4 identical layers
    assert hold[0] % 4 == 0 and per_layer > 0
    c = (need[:, None] - ov) // per_layer
    assert ((need[:, None] - ov) % per_layer == 0).all()
    assert c[0, 0] == 4                           # the value the paper prints
    assert np.array_equal(c[:, :4], gold)


# ------------------------------------------------------------------ P7: PP/TP merge rule as a closed form
@pytest.mark.parametrize("tp_old,tp_new,pp_old,pp_new", [(2, 4, 4, 2), (4, 2, 2, 4), (2, 2, 1, 4), (1, 4, 4, 4)])
def test_P7_pp_tp_merge_rule(tp_old, tp_new, pp_old, pp_new):
    """merged PP/TP cost = (#common layers) x (TP overlap fraction of the sharded part) + the
    replicated part — computed here from the logical tensor list alone."""
    model = dict(style=STYLE_GPT, n_layers=8, hidden=16, n_q_heads=4, n_kv_heads=4, head_dim=4, ffn_hidden=32,
                 vocab=16, max_pos=4, tied=0, param_bytes=2, kinds=0b1111)
    old = O.Layout(model, dict(tp=tp_old, pp=pp_old, dp=1, dist_opt=0))
    new = O.Layout(model, dict(tp=tp_new, pp=pp_new, dp=1, dist_opt=0))
    ov, need, hold = O.overlap(old, new, only_layers=True)
    lts = O.logical_tensors(model)
    sharded = sum(r * c for r, c, split, where, layer in lts if where == 1 and layer == 0 and split != 0)
    repl = sum(r * c for r, c, split, where, layer in lts if where == 1 and layer == 0 and split == 0)
    bytes_per_elem = sum(O.kind_bytes(model, k) for k in range(4))
    lcm = np.lcm(tp_old, tp_new)
    for n in range(new.n_dev):
        rn, sn = n % tp_new, n // tp_new
        for o in range(old.n_dev):
            ro, so = o % tp_old, o // tp_old
            ln = set(range(sn * 8 // pp_new, (sn + 1) * 8 // pp_new))
            lo = set(range(so * 8 // pp_old, (so + 1) * 8 // pp_old))
            un = set(range(rn * lcm // tp_new, (rn + 1) * lcm // tp_new))      # LCM units
            uo = set(range(ro * lcm // tp_old, (ro + 1) * lcm // tp_old))
            expect = len(ln & lo) * (sharded * len(un & uo) // lcm + repl) * bytes_per_elem
            assert ov[n, o] == expect, (n, o)


# ------------------------------------------------------------------ survey cross-check values (independent calculator)
@pytest.mark.parametrize("row", read_golden("survey_scratch_bytes.txt"), ids=lambda r: r[0])
def test_P11_survey_scratch_bytes(row):
    name, s_hold, s_need, local, remote = row[0], *map(int, row[1:])
    w = workload(name)
    old, new = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    ov, need, hold = O.overlap(old, new, method="ranges")
    if s_hold >= 0:
        assert hold.sum() == s_hold and need.sum() == s_need
    _, val = O.sketch_hungarian(ov)
    assert val == local and need.sum() - val == remote


def test_P11_closed_forms_bounds_attained():
    """local*(pi) <= min(sum need, sum hold) always; c1 attains sum hold, c2 and c5b attain sum need (all local)."""
    for name, which in (("c1", "hold"), ("c2", "need"), ("c5b", "need")):
        w = workload(name)
        old, new = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
        ov, need, hold = O.overlap(old, new, method="ranges")
        _, val = O.sketch_hungarian(ov)
        assert val <= min(need.sum(), hold.sum())
        assert val == (hold.sum() if which == "hold" else need.sum())
    # c5b structure: overlap[n][o] = need[n] where stage and TP rank match (any DP pair); only the TP-replicated
    # norm weights where the stage matches but the TP rank differs; 0 across stages
    tp, dpo, dpn = 8, 4, 3
    for n in range(0, new.n_dev, 7):
        rn, sn = n % tp, n // (tp * dpn)
        for o in range(old.n_dev):
            ro, so = o % tp, o // (tp * dpo)
            if sn != so:
                assert ov[n, o] == 0
            elif rn == ro:
                assert ov[n, o] == need[n]
            else:
                assert 0 < ov[n, o] < need[n] // 100


def test_ranges_routine_matches_elementwise():
    for name in ("c1", "s2", "s3", "s4", "s4odd", "s5"):
        w = workload(name)
        old, new = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
        a = O.overlap(old, new, method="elementwise")
        b = O.overlap(old, new, method="ranges")
        for x, y in zip(a, b):
            assert np.array_equal(x, y), name


# ------------------------------------------------------------------ P5/P6: sketch
def test_P5_P6_hungarian_vs_bruteforce_vs_scipy():
    from scipy.optimize import linear_sum_assignment       # the routine the paper calls
    rng = np.random.default_rng(7)
    for trial in range(60):
        P = int(rng.integers(1, 8)); n = int(rng.integers(1, P + 1))
        kind = trial % 3
        if kind == 0:
            ov = rng.integers(0, 1000, size=(n, P))
        elif kind == 1:
            ov = rng.integers(0, 3, size=(n, P)) * 10**11          # heavy ties, large values
        else:
            ov = np.zeros((n, P), np.int64); ov[:, : max(1, P // 2)] = rng.integers(0, 50, size=(n, max(1, P // 2)))
        ov = ov.astype(np.int64)
        mb, vb, cnt = O.sketch_bruteforce(ov)
        mh, vh = O.sketch_hungarian(ov)
        r, c = linear_sum_assignment(ov, maximize=True)
        assert cnt == np.prod([P - i for i in range(n)])             # every injective map was tried
        assert vb == vh == int(ov[r, c].sum())
        assert len(set(mh.tolist())) == n and sum(int(ov[i, mh[i]]) for i in range(n)) == vh
        # with an availability mask (preemption, A18)
        avail = (rng.random(P) < 0.8).astype(np.uint8)
        if avail.sum() >= n:
            mb2, vb2, _ = O.sketch_bruteforce(ov, avail)
            mh2, vh2 = O.sketch_hungarian(ov, avail)
            assert vb2 == vh2 and all(avail[p] for p in mh2)


def test_P6_scipy_on_config_matrices():
    from scipy.optimize import linear_sum_assignment
    for name in ("c3", "c4", "c5b"):
        w = workload(name)
        old, new = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
        ov, _, _ = O.overlap(old, new, method="ranges")
        r, c = linear_sum_assignment(ov, maximize=True)
        m, v = O.sketch_hungarian(ov)
        assert v == int(ov[r, c].sum())
        assert len(set(m.tolist())) == new.n_dev


# ------------------------------------------------------------------ P2-P4, P8-P10 on one reconfiguration
def _check_reconfiguration(model, old_cfg, new_cfg, seed, device_map=None, payload="stamp"):
    old, new = _layouts(model, old_cfg, new_cfg)
    if old is None:
        return False
    P = O.P_of(old, new)
    ov, need, hold = O.overlap(old, new)
    lts = O.logical_tensors(model)
    # --- P3 sum identities with replication factors (per element: KV-head replication makes them vary inside a tensor)
    def weighted(layout_mine, dev, layout_other):
        tot = 0
        for k in layout_mine.kinds():
            lt, _, row, col = layout_mine.global_of(dev, k)
            for t in np.unique(lt):
                sel = lt == t
                tot += int(replication_map(layout_other, k, lts, int(t))[row[sel], col[sel]].sum()) * O.kind_bytes(model, k)
        return tot
    for n in range(new.n_dev):
        assert ov[n].sum() == weighted(new, n, old), ("row sum", n)
    for o in range(old.n_dev):
        assert ov[:, o].sum() == weighted(old, o, new), ("col sum", o)
    assert (ov <= need[:, None]).all() and (ov <= hold[None, :]).all()
    # --- P5 sketch
    if device_map is None:
        if P <= 7:
            device_map, val, _ = O.sketch_bruteforce(ov)
            _, vh = O.sketch_hungarian(ov)
            assert vh == val
        else:
            device_map, val = O.sketch_hungarian(ov)
    # --- migrate with index-stamped logical payload (P8) and P4 reassembly
    logical = make_logical(model, seed, "stamp" if payload == "stamp" else "values")
    src = shard_all(old, logical)
    dst, T, ovr = O.migrate(old, new, device_map, src, want_overrides=True)
    for n in range(new.n_dev):
        for k in new.kinds():
            assert np.array_equal(dst[(n, k)], new.shard_from_logical(n, k, logical[k])), ("P8", n, k)
    rebuilt, cover, consistent = reassemble(new, dst, logical)
    assert consistent
    for k in logical:
        for t in range(len(lts)):
            assert np.array_equal(rebuilt[k][t], logical[k][t]), ("P4", k, t)
            assert np.array_equal(cover[k][t], replication_map(new, k, lts, t)), ("P4 cover", k, t)
    # --- P3 on T
    for n in range(new.n_dev):
        assert T[:, device_map[n]].sum() == need[n]
    assert T.sum() == need.sum()
    local = sum(int(T[device_map[n], device_map[n]]) for n in range(new.n_dev))
    assert local == sum(int(ov[n, device_map[n]]) for n in range(new.n_dev))      # local-first keeps overlap local
    # --- P9 replica-stamped payload: the values name the source, the histogram is T.  orc_migrate and orc_source_of share
    # the rule's code (orc_pick_source), so this block checks their CONSISTENCY and the histogram identity only; the rule
    # itself is pinned by re-deriving every source from holders_of in test_megatron_geometry_pins.py
    # (test_sources_rederived_from_holders) and, under failure masks, in test_failure_pins.py
    stamps = stamp_all(old)
    dst2, T2, _ = O.migrate(old, new, device_map, stamps)
    hist = np.zeros_like(T)
    for n in range(new.n_dev):
        for k in new.kinds():
            cnt = new.buffer_elems(n, k)
            if cnt == 0:
                continue
            sd, sl = O.source_of(old, new, device_map, n, k, np.arange(cnt))
            es = new.elem_bytes(k)
            for o in np.unique(sd):
                sel = sd == o
                exp = position_stamp(int(o), k, old.buffer_elems(int(o), k), es)[sl[sel]]
                assert np.array_equal(dst2[(n, k)][sel], exp), ("P9", n, k, o)
                hist[o, device_map[n]] += int(sel.sum()) * es
    assert np.array_equal(hist, T) and np.array_equal(T2, T)
    # --- P10 exactly once
    for n in range(new.n_dev):
        for k in new.kinds():
            cnt = new.buffer_elems(n, k)
            written = np.zeros(cnt, np.uint8)
            O.migrate_range(old, new, device_map, n, k, 0, cnt, None, None, None, written)
            assert (written == 1).all()
    return True


def test_P2_identity_reconfiguration():
    for name, model in tiny_models():
        for cfg in (dict(tp=2, pp=2, dp=2, dist_opt=1), dict(tp=2, pp=2, dp=1, dist_opt=0)):
            old, new = _layouts(model, cfg, cfg)
            if old is None:
                continue
            ov, need, hold = O.overlap(old, new)
            ident = np.arange(new.n_dev, dtype=np.int32)
            assert np.array_equal(np.diag(ov), need) and np.array_equal(need, hold)
            logical = make_logical(model, 11)
            src = shard_all(old, logical)
            dst, T, _ = O.migrate(old, new, ident, src)
            assert np.array_equal(T, np.diag(need))                      # Refer only: nothing moves
            for key in src:
                assert np.array_equal(src[key], dst[key])
            _, v = O.sketch_hungarian(ov)
            assert v == need.sum()


def test_config1_full_pins():
    w = workload("c1")
    assert _check_reconfiguration(w["model"], w["old"], w["new"], w["seed"], payload="values")


@pytest.mark.parametrize("name", ["s2", "s4odd", "s5b_small"])
def test_scaled_pins(name):
    if name == "s5b_small":
        w = workload("s5b")
        w["old"], w["new"] = dict(tp=2, pp=4, dp=4, dist_opt=0), dict(tp=2, pp=4, dp=3, dist_opt=0)
        w["model"].update(n_layers=4, n_kv_heads=2, n_q_heads=4, head_dim=16)
    else:
        w = workload(name)
    assert _check_reconfiguration(w["model"], w["old"], w["new"], w["seed"])


def test_config3_row_sum_identity_when_no_override():
    """P3 (config 3 shape): TP and DP unchanged => A6(ii) is a bijection between replicas; when local-first never
    overrides the designated holder, every old device sends exactly what it holds... only for devices whose
    content is still needed: sum_p T[o][p] <= hold[o], with equality summed over all o iff nothing is dropped."""
    w = workload("s3")
    old, new = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    ov, need, hold = O.overlap(old, new)
    m, v = O.sketch_hungarian(ov)
    _, T, overrides = O.migrate(old, new, m, None, want_overrides=True)
    assert overrides == 0
    assert (T.sum(axis=1) <= hold).all()
    assert T.sum() == need.sum() == hold.sum()          # same replication on both sides, nothing dropped
    assert np.array_equal(T.sum(axis=1), hold)


def _sweep_pairs():
    cfgs = tiny_parallel_cfgs(max_devices=8)
    pairs = list(itertools.product(range(len(cfgs)), repeat=2))
    rng = np.random.default_rng(2607_04749)
    out = []
    for mi, (name, model) in enumerate(tiny_models()):
        pick = rng.choice(len(pairs), size=36, replace=False)
        for pi in pick:
            a, b = pairs[pi]
            out.append((name, cfgs[a], cfgs[b]))
    return out


def test_P12_swept_tiny_layouts():
    ran = 0
    for i, (name, a, b) in enumerate(_sweep_pairs()):
        if _check_reconfiguration(TINY[name], a, b, 100 + i):
            ran += 1
    assert ran >= 60


def test_P12_scale_in_with_avail_mask_and_arbitrary_maps():
    """Any injective map (not only the optimum) must migrate correctly, incl. onto fresh devices (A18)."""
    rng = np.random.default_rng(5)
    model = TINY["gpt_t"]
    a, b = dict(tp=2, pp=2, dp=1, dist_opt=0), dict(tp=1, pp=4, dp=2, dist_opt=1)      # 4 -> 8 (scale out)
    for _ in range(3):
        dm = rng.permutation(8).astype(np.int32)
        assert _check_reconfiguration(model, a, b, 9, device_map=dm)
    a, b = dict(tp=2, pp=2, dp=2, dist_opt=1), dict(tp=2, pp=1, dp=1, dist_opt=0)      # 8 -> 2 (scale in)
    for _ in range(3):
        dm = rng.permutation(8)[:2].astype(np.int32)
        assert _check_reconfiguration(model, a, b, 9, device_map=dm)
