"""-m gpu parity of state chunking (f2): a kind-major plan cut into rounds of bounded staging must
write exactly what the element-wise oracle writes, while only the current kind's buffers exist (eager release of the
source side, on-demand allocation of the destination side)."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload, tiny_models
from oracle import oracle as O
from helpers import make_logical, shard_all, sharded_payload, oracle_migrate
from gpu_helpers import upload, download


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _run_rounds(E, model, old_cfg, new_cfg, seed, cap, flags, device_map=None, poison=0x5A):
    oo, on = O.Layout(model, old_cfg), O.Layout(model, new_cfg)
    src_np = sharded_payload(oo, seed, "stamp")
    old, new = E.etc_layout_create(model, old_cfg), E.etc_layout_create(model, new_cfg)
    if device_map is None:
        ov, _, _ = E.etc_cost_matrix(old, new)
        dm, _ = E.etc_sketch(ov)
    else:
        dm = torch.tensor(np.asarray(device_map, np.int32)).cuda()
    plan = E.etc_plan_create(old, new, dm, flags | E.ETC_KIND_MAJOR)
    rounds = E.etc_plan_set_rounds(plan, cap)
    st = plan.stats
    # bookkeeping of the rounds
    assert all(r.staging_bytes <= cap for r in rounds)
    assert sum(r.staged_bytes for r in rounds) == st.staged_bytes
    assert sum(r.local_bytes for r in rounds) == st.local_bytes + st.remote_bytes - st.staged_bytes
    assert sum(r.n_chunks_staged for r in rounds) == st.n_chunks_staged
    assert sum(r.n_chunks_local for r in rounds) == st.n_chunks_local
    kinds = [r.kind for r in rounds]
    assert kinds == sorted(kinds)
    for r in rounds:
        assert 0 <= r.sub < r.n_sub
    staging = torch.full((max(max((r.staging_bytes for r in rounds), default=0), 16),), poison, dtype=torch.uint8,
                         device="cuda")
    out = {}
    peak_live = 0
    for k in sorted(set(kinds)):
        # on-demand: only kind k's buffers exist while its rounds run
        src_k = upload({key: v for key, v in src_np.items() if key[1] == k})
        dst_k = {key: v for key, v in E.alloc_buffers(new, fill=poison).items() if key[1] == k}
        for i, r in enumerate(rounds):
            if r.kind != k:
                continue
            staging.fill_(poison)                                  # nothing may survive from the previous round
            E.etc_migrate_round(plan, i, src_k, dst_k, staging)
        torch.cuda.synchronize()
        es = 4 if k else model["param_bytes"]
        for key, t in dst_k.items():
            out[key] = download(t, es)
        del src_k, dst_k                                           # eager release
    dst, T, _ = oracle_migrate(oo, on, dm.cpu().numpy(), src_np)
    assert np.array_equal(plan.traffic(), T)
    for key, exp in dst.items():
        if exp.shape[0] == 0:
            continue
        assert np.array_equal(out[key], exp), (key, int((out[key] != exp).sum()))
    return plan, rounds


@pytest.mark.parametrize("name", ["c1", "s2", "s2odd", "s3", "s4", "s4odd", "s5"])
@pytest.mark.parametrize("cap", [2 * 65536, 1 << 20, 1 << 34])
def test_rounds_vs_oracle(E, name, cap):
    w = workload(name)
    for flags in (0, 1):
        plan, rounds = _run_rounds(E, w["model"], w["old"], w["new"], w["seed"], cap, flags)
        if cap == 1 << 34:
            assert all(r.n_sub == 1 for r in rounds)               # one round per kind when staging is unbounded
    if cap == 2 * 65536 and name in ("s3", "s5"):
        assert max(r.n_sub for r in rounds) > 1                    # the small bound really cuts kinds into sub-rounds


def test_rounds_arbitrary_maps_and_reset(E):
    rng = np.random.default_rng(5)
    w = workload("s4")
    for _ in range(2):
        _run_rounds(E, w["model"], w["old"], w["new"], 9, 3 * 65536, 0, device_map=rng.permutation(32).astype(np.int32))
    # the bound can be changed on the same plan
    old, new = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    plan = E.etc_plan_create(old, new, np.arange(32, dtype=np.int32), E.ETC_KIND_MAJOR)
    a = E.etc_plan_set_rounds(plan, 2 * 65536)
    b = E.etc_plan_set_rounds(plan, 1 << 30)
    assert len(a) > len(b) and len(b) == len(set(r.kind for r in b))


def test_rounds_errors(E):
    model = dict(tiny_models())["gpt_t"]
    a, b = dict(tp=2, pp=1, dp=1, dist_opt=0), dict(tp=1, pp=2, dp=1, dist_opt=0)
    old, new = E.etc_layout_create(model, a), E.etc_layout_create(model, b)
    plain = E.etc_plan_create(old, new, np.arange(2, dtype=np.int32), 0)
    with pytest.raises(E.EtcError) as e:
        E.etc_plan_set_rounds(plain, 1 << 20)                      # not kind-major
    assert e.value.code == -1
    km = E.etc_plan_create(old, new, np.arange(2, dtype=np.int32), E.ETC_KIND_MAJOR)
    with pytest.raises(E.EtcError):
        E.etc_plan_set_rounds(km, 65536)                           # bound below two chunks
    rounds = E.etc_plan_set_rounds(km, 1 << 20)
    src, dst = E.alloc_buffers(old), E.alloc_buffers(new)
    stg = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    assert E.lib().etc_migrate_round(km.h, len(rounds), None, None, None, 3, None) == -1   # no such round
    k0 = rounds[0].kind
    src_missing = {key: v for key, v in src.items() if key[1] != k0}
    with pytest.raises(E.EtcError):                                # the round's own kind must be present
        E.etc_migrate_round(km, 0, src_missing, dst, stg)
