"""-m "not gpu": pins of oracle/defrag.py (Algorithm 2 + coalescing) against things other than itself:
hand-worked examples (tests/golden/defrag_handworked.txt), closed forms and invariants from the prose, and the traffic
inequality that communication coalescing guarantees."""
from __future__ import annotations
import os
import numpy as np
import pytest

from helpers import GOLDEN
from oracle import defrag as D
from oracle import oracle as O
from etc_inputs import tiny_models, workload


def _parse():
    cases = []
    for line in open(os.path.join(GOLDEN, "defrag_handworked.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        head, dm, mo, final = [x.strip() for x in line.split(";")]
        mode, pw, cw, n = head.split()
        ops = [tuple(int(v) for v in t.split(":")) for t in mo.split()]
        cases.append((mode, int(pw), int(cw), int(n), [int(x) for x in dm.split()], ops, [int(x) for x in final.split()]))
    return cases


@pytest.mark.parametrize("case", _parse(), ids=lambda c: f"{c[0]}-{c[1]}to{c[2]}-n{c[3]}")
def test_handworked_examples(case):
    mode, pw, cw, n, dm, ops, final = case
    if mode == "occupancy":
        mo = D.defragmentation_for_occupancy(pw, cw, dm, n)
        assert mo == ops
        assert D.apply_occupancy(dm, mo) == final
    else:
        mo = D.defragmentation_for_efficiency(pw, cw, dm, n)
        assert mo == ops
        assert D.apply_efficiency(dm, mo) == final
    assert D.defragment(pw, cw, dm, n, mode) == (final, len(ops))


def _random_maps(rng, pw, cw, count):
    P = max(pw, cw)
    for _ in range(count):
        yield [int(x) for x in rng.permutation(P)[:cw]]


def test_occupancy_closed_forms():
    """idle devices in order are paired with occupied devices in reverse order until they meet.  Hence
    (a) afterwards the occupied devices are exactly [0, cw) — whole nodes at the end are freed; (b) a rank that already
    sat inside [0, cw) did not move; (c) #operators == #idle devices below cw == #occupied devices at or above cw;
    (d) the k-th operator pairs the k-th lowest idle device with the k-th highest occupied device."""
    rng = np.random.default_rng(7)
    for pw, cw, n in [(8, 4, 4), (16, 12, 4), (12, 5, 2), (32, 8, 8), (9, 9, 3), (4, 8, 4), (64, 48, 8)]:
        for dm in _random_maps(rng, pw, cw, 40):
            mo = D.defragmentation_for_occupancy(pw, cw, dm, n)
            out = D.apply_occupancy(dm, mo)
            assert sorted(out) == list(range(cw))                                           # (a)
            for r in range(cw):
                if dm[r] < cw:
                    assert out[r] == dm[r]                                                  # (b)
            occupied = set(dm)
            idle_below = [d for d in range(cw) if d not in occupied]
            occ_above = sorted((d for d in occupied if d >= cw), reverse=True)
            assert len(mo) == len(idle_below) == len(occ_above)                             # (c)
            assert mo == list(zip(idle_below, occ_above))                                   # (d)


def test_efficiency_closed_forms():
    """afterwards every node's load equals its target (rank k on device k, so every TP group of size
    <= n that divides n sits inside one node); every operator names a device whose load differed from its target."""
    rng = np.random.default_rng(11)
    for pw, cw, n in [(8, 8, 4), (12, 12, 4), (16, 12, 4), (8, 4, 4), (6, 6, 2), (4, 8, 4), (64, 64, 8)]:
        P = max(pw, cw)
        for t in range(40):
            dm = list(range(cw))
            if t:                                             # fragment a few nodes only
                for _ in range(int(rng.integers(1, 4))):
                    a, b = rng.integers(0, cw, 2)
                    dm[a], dm[b] = dm[b], dm[a]
                if t % 3 == 0:
                    dm = [int(x) for x in rng.permutation(P)[:cw]]
            mo = D.defragmentation_for_efficiency(pw, cw, dm, n)
            out = D.apply_efficiency(dm, mo)
            assert out == list(range(cw))
            p2c = D.p2c_from_device_map(dm, P)
            for pProc, cProc in mo:
                assert p2c[pProc] == cProc and pProc != cProc
            assert len(mo) == sum(1 for r in range(cw) if p2c[r] != r)
            for g in range(cw // n):                          # TP groups of n consecutive ranks: one node each
                assert len({out[r] // n for r in range(g * n, (g + 1) * n)}) == 1


def _remote_bytes(oo, on, dm):
    _, T, _ = O.migrate(oo, on, np.asarray(dm, np.int32), None)
    return int(T.sum() - np.trace(T)), T


@pytest.mark.parametrize("mode", ["occupancy", "efficiency", "both"])
def test_coalescing_never_moves_more_than_two_stages(mode):
    """migration i->k followed by de-fragmentation k->j is coalesced into i->j.  Two-stage traffic =
    remote(pi) + sum of need[rank] over re-placed ranks (stage 2 ships the whole rank state); the coalesced plan ships
    remote(pi') bytes.  Coalescing must never move more, and each rank still receives exactly need[n] bytes."""
    _, model = tiny_models()[0]
    cases = [((1, 4, 1), (1, 2, 1), 2), ((2, 4, 1), (2, 2, 1), 4), ((2, 2, 2), (4, 2, 1), 4), ((1, 2, 2), (2, 2, 1), 2),
             ((2, 2, 1), (2, 4, 1), 4)]
    for old_c, new_c, n in cases:
        oc = dict(tp=old_c[0], pp=old_c[1], dp=old_c[2], dist_opt=0)
        nc = dict(tp=new_c[0], pp=new_c[1], dp=new_c[2], dist_opt=0)
        oo, on = O.Layout(model, oc), O.Layout(model, nc)
        ov, need, hold = O.overlap(oo, on)
        dm, _ = O.sketch_hungarian(ov)
        final, ops = D.defragment(oo.n_dev, on.n_dev, dm, n, mode)
        r0, _ = _remote_bytes(oo, on, dm)
        r1, T1 = _remote_bytes(oo, on, final)
        moved = [r for r in range(on.n_dev) if final[r] != dm[r]]
        two_stage = r0 + int(sum(need[r] for r in moved))
        assert r1 <= two_stage
        for r in range(on.n_dev):
            assert int(T1[:, final[r]].sum()) == int(need[r])
        if not moved:
            assert r1 == r0


def test_c3_preemption_shape_frees_whole_nodes():
    """BASELINE.json configs[2] (16 -> 12 devices, nodes of 4): after occupancy-level remapping one whole node is idle."""
    w = workload("c3")
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    ov, need, hold = O.overlap(oo, on, method="ranges")
    dm, _ = O.sketch_hungarian(ov)
    final, ops = D.defragment(16, 12, dm, 4, "occupancy")
    assert sorted(final) == list(range(12))
    assert {d // 4 for d in final} == {0, 1, 2}
