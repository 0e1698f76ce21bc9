"""-m "not gpu": pin of the oracle's source rule for DP growth against the paper's statement: "When
increasing DP size during reconfiguration ... each PP/TP process in existing DP groups sends all model states to its
counterpart in new DP groups.  And the source groups are selected in a round-robin manner to ensure the load balance
among existing DP groups."  With the PP/TP configuration unchanged, the existing DP groups kept in place and the new
groups on fresh devices, the traffic matrix T has a closed form that does not come from the oracle:
  * new group d' >= dp_old on (s, r) receives its whole state from exactly one old device, the (s, r) process of
    old group d' mod dp_old (counterpart + round-robin);
  * old device (d, s, r) therefore sends hold[(d,s,r)] x #{d' in [dp_old, dp_new): d' mod dp_old == d} bytes, so the
    per-group send counts differ by at most one state (load balance), and are all equal when dp_old divides dp_new."""
from __future__ import annotations
import numpy as np
import pytest

from etc_inputs import tiny_models
from oracle import oracle as O

MODELS = dict(tiny_models())


def _cfg(tp, pp, dp, dist_opt=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt)


def _dev(cfg, d, s, r):
    return r + cfg["tp"] * (d + cfg["dp"] * s)


def growth_map(old_c, new_c):
    """existing DP groups stay on their devices, new groups go to fresh devices [n_old, n_new) in rank order"""
    n_old = old_c["tp"] * old_c["pp"] * old_c["dp"]
    dm, fresh = [], n_old
    for n in range(new_c["tp"] * new_c["pp"] * new_c["dp"]):
        r, d, s = n % new_c["tp"], (n // new_c["tp"]) % new_c["dp"], n // (new_c["tp"] * new_c["dp"])
        if d < old_c["dp"]:
            dm.append(_dev(old_c, d, s, r))
        else:
            dm.append(fresh); fresh += 1
    return np.asarray(dm, np.int32)


def closed_form_T(old_c, new_c, hold, dm):
    n_old = len(hold)
    P = max(n_old, len(dm))
    T = np.zeros((P, P), np.int64)
    for n, p in enumerate(dm):
        r, d, s = n % new_c["tp"], (n // new_c["tp"]) % new_c["dp"], n // (new_c["tp"] * new_c["dp"])
        src = _dev(old_c, d % old_c["dp"], s, r)                # counterpart in group d' mod dp_old
        T[src, p] += hold[src]
    return T


@pytest.mark.parametrize("name,tp,pp,dp_old,dp_new", [("gpt_t", 2, 2, 1, 2), ("gpt_t", 1, 2, 2, 4), ("gpt_u", 2, 1, 2, 5),
                                                      ("llama_u", 2, 2, 2, 3), ("llama_t", 1, 2, 3, 8), ("gpt_np", 2, 2, 1, 4)])
def test_dp_growth_round_robin_balance(name, tp, pp, dp_old, dp_new):
    model = MODELS[name]
    old_c, new_c = _cfg(tp, pp, dp_old), _cfg(tp, pp, dp_new)
    oo, on = O.Layout(model, old_c), O.Layout(model, new_c)
    ov, need, hold = O.overlap(oo, on)
    dm = growth_map(old_c, new_c)
    # the growth map is an optimal sketch: every existing group keeps its whole state local
    assert sum(int(ov[n, dm[n]]) for n in range(on.n_dev)) == O.sketch_hungarian(ov)[1] == int(hold[:oo.n_dev].sum())
    _, T, _ = O.migrate(oo, on, dm, None)
    assert np.array_equal(T, closed_form_T(old_c, new_c, hold, dm))
    # load balance among the existing DP groups: whole states sent by each group
    sent = np.zeros(dp_old, np.int64)
    for o in range(oo.n_dev):
        d = (o // tp) % dp_old
        off = int(T[o].sum() - T[o, o])
        assert off % int(hold[o]) == 0
        sent[d] += off // int(hold[o])
    per_group = sent // (tp * pp)
    assert (sent % (tp * pp) == 0).all() and per_group.sum() == dp_new - dp_old
    assert per_group.max() - per_group.min() <= 1
    if dp_new % dp_old == 0:
        assert (per_group == dp_new // dp_old - 1).all()
