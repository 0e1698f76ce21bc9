"""-m "not gpu": the oracle's sketch objective against Algorithm 1 AS PRINTED, run with the very
routine the paper calls (SciPy's linear_sum_assignment): cost c[n][o] = need[n] - overlap[n][o],
zero-padded to k x k (line 3), solved for MINIMUM cost (line 5), pairs touching the padding dropped (lines 6-8).
  * M <= N (no new rank lands on a padded column): the printed algorithm and the oracle's "maximise the bytes that stay
    local" have the same optimum (reading A4: min sum(need - overlap) = sum(need) - max sum(overlap));
  * M > N (scale-out): a padded column costs 0 instead of need[n], so the printed algorithm prefers to leave the ranks
    with the LARGEST need on fresh devices; it can never keep more bytes local than the oracle's optimum, and on a
    layout with unequal needs (first / last pipeline stage carry the embeddings) it keeps strictly fewer: the reason
    for reading A4."""
from __future__ import annotations
import numpy as np
import pytest

scipy_opt = pytest.importorskip("scipy.optimize")

from etc_inputs import tiny_models, workload
from oracle import oracle as O

MODELS = dict(tiny_models())


def algorithm1_as_printed(ov, need, n_old):
    """returns (pairs kept, local bytes they keep)"""
    M, N = ov.shape[0], n_old
    k = max(M, N)
    C = np.zeros((k, k), np.int64)
    C[:M, :N] = need[:, None] - ov[:, :N]
    rows, cols = scipy_opt.linear_sum_assignment(C)
    pairs = [(i, j) for i, j in zip(rows, cols) if i < M and j < N]
    return pairs, int(sum(ov[i, j] for i, j in pairs))


def _cfg(tp, pp, dp, dist_opt=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt)


@pytest.mark.parametrize("name,a,b", [("gpt_t", _cfg(2, 2, 1), _cfg(1, 2, 2)), ("gpt_u", _cfg(2, 2, 2), _cfg(4, 2, 1)),
                                      ("llama_u", _cfg(4, 1, 2), _cfg(2, 2, 1)), ("gpt_np", _cfg(1, 4, 2), _cfg(2, 2, 1)),
                                      ("llama_t", _cfg(2, 2, 2), _cfg(1, 2, 2, 1))])
def test_printed_algorithm_equals_oracle_when_no_padding_is_used(name, a, b):
    m = MODELS[name]
    oo, on = O.Layout(m, a), O.Layout(m, b)
    assert on.n_dev <= oo.n_dev
    ov, need, hold = O.overlap(oo, on)
    pairs, local = algorithm1_as_printed(ov, need, oo.n_dev)
    assert len(pairs) == on.n_dev                                   # every curr rank is paired with a real prev rank
    assert local == O.sketch_hungarian(ov)[1]
    if ov.shape[1] <= 8:
        assert local == O.sketch_bruteforce(ov)[1]


def test_named_configs_c1_c2_c3():
    for name in ("c1", "c2", "c3"):
        w = workload(name)
        oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
        ov, need, hold = O.overlap(oo, on, method="ranges")
        pairs, local = algorithm1_as_printed(ov, need, oo.n_dev)
        assert local == O.sketch_hungarian(ov)[1]


def test_printed_objective_is_blind_on_scale_out_with_unequal_needs():
    """PP2 -> PP4 with untied embeddings, TP = DP = 1: 2 old devices, 4 new ranks; ranks 0 and 3 carry the embeddings and
    need the most.  Every curr rank either fits its prev device entirely (cost 0) or sits on a padded column (cost 0):
    the printed objective is 0 for assignments that keep very different numbers of bytes in place, so which one SciPy
    returns is an accident of tie-breaking; the oracle's objective separates them."""
    import itertools
    m = dict(MODELS["llama_u"], vocab=64)
    oo, on = O.Layout(m, _cfg(1, 2, 1)), O.Layout(m, _cfg(1, 4, 1))
    ov, need, hold = O.overlap(oo, on)
    assert need[0] > need[1] and need[3] > need[2]
    C = np.zeros((4, 4), np.int64)
    C[:, :2] = need[:, None] - ov[:, :2]
    by_cost = {}
    for perm in itertools.permutations(range(4)):
        cost = int(sum(C[i, perm[i]] for i in range(4)))
        local = int(sum(ov[i, perm[i]] for i in range(4) if perm[i] < 2))
        by_cost.setdefault(cost, set()).add(local)
    best_cost = min(by_cost)
    assert best_cost == 0 and len(by_cost[0]) > 1                   # several optima of the printed objective ...
    best = O.sketch_bruteforce(ov)[1]
    assert max(by_cost[0]) == best and min(by_cost[0]) < best       # ... only one of which keeps the most bytes local
    pairs, local = algorithm1_as_printed(ov, need, oo.n_dev)
    assert local in by_cost[0] and local <= best
    # never better than the oracle's optimum, on any scale-out
    for name, a, b in [("gpt_t", _cfg(1, 2, 1), _cfg(2, 2, 1)), ("llama_u", _cfg(2, 1, 1), _cfg(2, 2, 2)), ("gpt_np", _cfg(1, 1, 2), _cfg(2, 2, 1))]:
        lo, ln = O.Layout(MODELS[name], a), O.Layout(MODELS[name], b)
        v, nd, _ = O.overlap(lo, ln)
        assert algorithm1_as_printed(v, nd, lo.n_dev)[1] <= O.sketch_hungarian(v)[1]
