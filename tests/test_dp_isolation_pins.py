"""-m "not gpu": pins of the oracle's DP-isolated cost matrix, the paper's own treatment of the DP dimension
("we isolate the PP/TP processes under different DP ranks ... the difference between the workloads to be
infinite"; ":179 the migration sketch within existing DP group is identical"; reading A5):
  * SURVEY.md 8(c) A5 [scratch], computed at survey time by a separate calculator: on config 2 the full matrix keeps
    5 798 395 904 B local, the DP-isolated formulation 2 899 197 952 B;
  * with the DP size unchanged, the isolated problem is dp independent copies of the dp = 1 problem (the paper's
    "migration of PP/TP processes is completely identical" among replicas): optimum = dp x the optimum of the dp = 1
    reconfiguration, solved separately;
  * a cell survives the mask iff the two DP ranks, recomputed here from the device id formula of reading A9, agree."""
from __future__ import annotations
import numpy as np
import pytest

from etc_inputs import tiny_models, workload
from oracle import oracle as O

MODELS = dict(tiny_models())


def _cfg(tp, pp, dp, dist_opt=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt)


def test_config2_isolated_optimum_is_half():
    w = workload("c2")
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    ov, need, hold = O.overlap(oo, on, method="ranges")
    assert O.sketch_hungarian(ov)[1] == 5798395904                         # SURVEY.md A5 [scratch]: full matrix
    iso = O.mask_cross_dp(oo, on, ov)
    assert O.sketch_hungarian(iso)[1] == 2899197952                        # SURVEY.md A5 [scratch]: DP-isolated
    assert O.sketch_hungarian(iso)[1] * 2 == int(need.sum())


@pytest.mark.parametrize("name,a,b,dp", [("gpt_t", (2, 2), (1, 2), 2), ("gpt_u", (1, 2), (2, 1), 3), ("llama_u", (2, 1), (1, 2), 2),
                                         ("gpt_np", (2, 2), (2, 1), 2), ("llama_t", (1, 2), (2, 2), 2)])
def test_isolated_problem_is_dp_copies_of_the_single_replica_problem(name, a, b, dp):
    m = MODELS[name]
    one = O.sketch_hungarian(O.overlap(O.Layout(m, _cfg(a[0], a[1], 1)), O.Layout(m, _cfg(b[0], b[1], 1)))[0])[1]
    oo, on = O.Layout(m, _cfg(a[0], a[1], dp)), O.Layout(m, _cfg(b[0], b[1], dp))
    ov, _, _ = O.overlap(oo, on)
    iso = O.mask_cross_dp(oo, on, ov)
    val = O.sketch_hungarian(iso)[1]
    assert val == dp * one
    if max(oo.n_dev, on.n_dev) <= 8:
        assert O.sketch_bruteforce(iso)[1] == val
    assert O.sketch_hungarian(ov)[1] >= val                                # isolation can only lose locality


def test_mask_keeps_exactly_the_same_dp_cells():
    for name, a, b in [("gpt_t", _cfg(2, 2, 2), _cfg(1, 2, 3)), ("llama_u", _cfg(1, 2, 4), _cfg(2, 2, 2)), ("gpt_u", _cfg(2, 1, 3, 1), _cfg(1, 1, 2))]:
        oo, on = O.Layout(MODELS[name], a), O.Layout(MODELS[name], b)
        ov, _, _ = O.overlap(oo, on)
        iso = O.mask_cross_dp(oo, on, ov)
        for n in range(on.n_dev):
            dn = (n // b["tp"]) % b["dp"]
            for o in range(ov.shape[1]):
                do = (o // a["tp"]) % a["dp"] if o < oo.n_dev else -1
                assert iso[n, o] == (ov[n, o] if do == dn else 0)
