"""-m "not gpu": pins of the oracle's failure-aware sourcing (f4; "Fault-tolerance through DP";
DESIGN.md reading A26) against things other than itself: the paper's d-1 guarantee, bit-identity with the failure-free
result (replicas are synchronized), sources re-derived from the independent holders_of enumeration, the
traffic identities, and the unrecoverable cases."""
from __future__ import annotations
import itertools
import numpy as np
import pytest

from etc_inputs import tiny_models, position_stamp
from oracle import oracle as O
from helpers import make_logical, shard_all, stamp_all

MODELS = dict(tiny_models())


def _cfg(tp, pp, dp, dist_opt=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt)


def _dev(cfg, d, s, r):
    return r + cfg["tp"] * (d + cfg["dp"] * s)


def _coords(cfg, dev):
    return (dev // cfg["tp"]) % cfg["dp"], dev // (cfg["tp"] * cfg["dp"]), dev % cfg["tp"]


CASES = [("gpt_t", _cfg(2, 2, 2), _cfg(1, 2, 2)), ("gpt_u", _cfg(1, 2, 4), _cfg(2, 1, 2)),
         ("llama_u", _cfg(2, 1, 4), _cfg(1, 2, 2)), ("gpt_np", _cfg(2, 2, 2), _cfg(2, 2, 3)),
         ("llama_t", _cfg(2, 2, 2), _cfg(2, 1, 4, 1))]


def _failure_sets(cfg, rng, count):
    """Random masks that keep at least one DP replica of every (stage, tp rank) alive (<= d-1 failures per group)."""
    n = cfg["tp"] * cfg["pp"] * cfg["dp"]
    out = []
    for _ in range(count):
        f = np.zeros(n, np.uint8)
        for s in range(cfg["pp"]):
            for r in range(cfg["tp"]):
                kill = rng.permutation(cfg["dp"])[: int(rng.integers(0, cfg["dp"]))]       # at most dp-1 of the group
                for d in kill:
                    f[_dev(cfg, int(d), s, r)] = 1
        out.append(f)
    return out


@pytest.mark.parametrize("name,old_c,new_c", CASES)
def test_d_minus_1_failures_are_survived_bit_identically(name, old_c, new_c):
    """"When the dimension of DP is d, ETC can accommodate at least d-1 hardware failures": with at least
    one surviving replica per (stage, tp rank) the migration succeeds, no byte is read from a failed device, and —
    replicas being synchronized — the new shards are bit-identical to the failure-free migration."""
    model = MODELS[name]
    rng = np.random.default_rng(hash(name) & 0xFFFF)
    oo, on = O.Layout(model, old_c), O.Layout(model, new_c)
    src = shard_all(oo, make_logical(model, 77, "stamp"))
    P = max(oo.n_dev, on.n_dev)
    _, need, _ = O.overlap(oo, on)
    for f in _failure_sets(old_c, rng, 6):
        dm = rng.permutation(P)[: on.n_dev].astype(np.int32)
        oo.set_failed(None)
        ref, T0, _ = O.migrate(oo, on, dm, src)
        oo.set_failed(f)
        poisoned = {k: (v if not f[k[0]] else np.full_like(v, 0xDEAD)) for k, v in src.items()}   # lost state
        got, T, _ = O.migrate(oo, on, dm, poisoned)
        for key in ref:
            assert np.array_equal(got[key], ref[key]), key
        assert T[: oo.n_dev][f.astype(bool), :].sum() == 0                      # nothing is read from a failed device
        for n in range(on.n_dev):
            assert int(T[:, dm[n]].sum()) == int(need[n])                       # each rank still receives need[n]
        if not f.any():
            assert np.array_equal(T, T0)
        ov, _, hold = O.overlap(oo, on)
        assert (ov[:, : oo.n_dev][:, f.astype(bool)] == 0).all() and (hold[: oo.n_dev][f.astype(bool)] == 0).all()
        oo.set_failed(None)
        ov0, _, hold0 = O.overlap(oo, on)
        alive = ~f.astype(bool)
        assert np.array_equal(ov[:, : oo.n_dev][:, alive], ov0[:, : oo.n_dev][:, alive])


def test_sources_match_rule_rederived_from_holders():
    """Reading A26 re-derived per element from the independent holders_of enumeration: (i) the destination device if
    it is alive and holds the element; (ii) else, among the alive holders with the designated stage and TP rank, the
    first in cyclic DP order starting at d' mod dp_old.  An element whose designated holder is alive keeps the source
    it has without failures."""
    model = MODELS["gpt_t"]
    old_c, new_c = _cfg(2, 2, 2), _cfg(1, 2, 2)
    oo, on = O.Layout(model, old_c), O.Layout(model, new_c)
    lts = O.logical_tensors(model)
    rng = np.random.default_rng(5)
    f = np.zeros(oo.n_dev, np.uint8); f[_dev(old_c, 0, 0, 1)] = 1; f[_dev(old_c, 1, 1, 0)] = 1
    dm = rng.permutation(8)[:4].astype(np.int32)
    oo.set_failed(None)
    base = {(n, k): O.source_of(oo, on, dm, n, k, np.arange(on.buffer_elems(n, k))) for n in range(4) for k in on.kinds()}
    oo.set_failed(f)
    for n in range(on.n_dev):
        d_new, s_new, r_new = _coords(new_c, n)
        p = int(dm[n])
        for k in on.kinds():
            cnt = on.buffer_elems(n, k)
            sd, sl = O.source_of(oo, on, dm, n, k, np.arange(cnt))
            lt, pc, row, col = on.global_of(n, k)
            for i in range(0, cnt, 7):
                holders = oo.holders_of(k, int(lt[i]), int(row[i]), int(col[i]))
                alive = [(dev, l) for dev, l in holders if not f[dev]]
                assert (int(sd[i]), int(sl[i])) in alive
                if any(dev == p for dev, _ in alive):
                    assert int(sd[i]) == p                                      # (i) local first
                    continue
                stages = sorted({_coords(old_c, dev)[1] for dev, _ in holders})
                s_des = stages[-1] if (pc[i] and len(stages) > 1) else stages[0]
                split = lts[int(lt[i])][2]
                cands = [(dev, l) for dev, l in holders if _coords(old_c, dev)[1] == s_des]
                if split == 0:                                                  # REPL over TP: r' mod tp_old
                    cands = [(dev, l) for dev, l in cands if _coords(old_c, dev)[2] == r_new % old_c["tp"]]
                order = [(d_new % old_c["dp"] + j) % old_c["dp"] for j in range(old_c["dp"])]
                pick = next(dev for d in order for dev, _ in cands if _coords(old_c, dev)[0] == d and not f[dev])
                assert int(sd[i]) == pick
                if not f[int(base[(n, k)][0][i])] and int(base[(n, k)][0][i]) != p:
                    assert int(sd[i]) == int(base[(n, k)][0][i])                # alive designated holder is kept


def test_position_stamps_never_name_a_failed_device():
    model = MODELS["llama_u"]
    old_c, new_c = _cfg(2, 1, 4), _cfg(1, 2, 2)
    oo, on = O.Layout(model, old_c), O.Layout(model, new_c)
    f = np.zeros(8, np.uint8); f[[0, 2, 4, 3]] = 1                              # r=0: d0,d1,d2 lost (d3 alive); r=1: d1 lost
    oo.set_failed(f)
    src = stamp_all(oo)
    dm = np.array([6, 7, 1, 5], np.int32)
    got, T, _ = O.migrate(oo, on, dm, src)
    for (n, k), buf in got.items():
        sd, sl = O.source_of(oo, on, dm, n, k, np.arange(buf.shape[0]))
        assert not f[sd].any()
        exp = np.zeros_like(buf)
        for o in np.unique(sd):
            sel = sd == o
            exp[sel] = position_stamp(int(o), k, oo.buffer_elems(int(o), k), on.elem_bytes(k))[sl[sel]]
        assert np.array_equal(buf, exp)
    assert T[[0, 2, 4, 3], :].sum() == 0


def test_unrecoverable_cases():
    """All d replicas of one (stage, tp rank) lost, or the single holder of a DP-sharded (dist-opt) range lost."""
    model = MODELS["gpt_t"]
    old_c, new_c = _cfg(2, 1, 2), _cfg(1, 1, 2)
    oo, on = O.Layout(model, old_c), O.Layout(model, new_c)
    f = np.zeros(4, np.uint8); f[_dev(old_c, 0, 0, 1)] = 1; f[_dev(old_c, 1, 0, 1)] = 1
    oo.set_failed(f)
    with pytest.raises(O.OracleError) as e:
        O.migrate(oo, on, np.array([0, 2], np.int32), None)
    assert e.value.code == -8
    f[:] = 0; f[_dev(old_c, 0, 0, 1)] = 1                                       # one replica left: fine
    oo.set_failed(f)
    O.migrate(oo, on, np.array([0, 2], np.int32), None)
    old_do = _cfg(2, 1, 2, 1)                                                   # dist-opt: MASTER/M/V ranges are unique
    od = O.Layout(model, old_do)
    od.set_failed(f)
    with pytest.raises(O.OracleError) as e:
        O.migrate(od, on, np.array([0, 2], np.int32), None)
    assert e.value.code == -8


def test_failed_device_reused_as_fresh_destination():
    """A failed device's slot may host a new rank (replaced hardware): it then holds nothing, so nothing is local."""
    model = MODELS["gpt_u"]
    old_c = new_c = _cfg(1, 2, 2)
    oo, on = O.Layout(model, old_c), O.Layout(model, new_c)
    src = shard_all(oo, make_logical(model, 3, "stamp"))
    f = np.zeros(4, np.uint8); f[1] = 1
    oo.set_failed(f)
    dm = np.arange(4, dtype=np.int32)                                           # identity: rank 1 sits on the failed slot
    got, T, _ = O.migrate(oo, on, dm, src)
    _, need, _ = O.overlap(oo, on)
    assert T[1, :].sum() == 0 and T[1, 1] == 0
    d1, s1, r1 = _coords(old_c, 1)
    twin = _dev(old_c, 1 - d1, s1, r1)
    assert T[twin, 1] == need[1]                                                # everything comes from its DP twin
    for key in got:
        assert np.array_equal(got[key], src[key])                               # identity reconfiguration, bit-exact
