"""-m gpu parity of the data path beyond 96 devices ("all devices emit their
instruction lists simultaneously", :382 bit-exact).

Up to 96 devices in all (384 buffer pointers) the copy kernels receive the shard pointers in their parameter block; beyond
that they read a pointer table in device memory that belongs to the plan (include/etc.h "Concurrency"), written on the
caller's stream before every launch — other template instances of the copy and zero-fill kernels, per-round tables for
etc_migrate_round.  BASELINE.json itself names a 512 -> 384-device reconfiguration, so that path must move bytes in a test:
  * s5b, the scaled twin of the 512 -> 384 layout (896 devices, 3584 pointers),
  * d64_128: 64 -> 128 devices, TP 4 -> 8, distributed optimizer on both sides, padded vocabulary that grows (zero-fill),
  * p64_128: 64 -> 128 devices small enough for an ETC_NO_SYNC plan to keep its counts on the device (bound-sized grids),
each through etc_plan_create + etc_migrate, etc_plan_set_rounds + etc_migrate_round, an ETC_NO_SYNC plan and
etc_migrate_state (row-maximum certificate, and a mask that defeats it so that the CTA Hungarian search decides), from
poisoned destination and staging buffers, compared byte for byte with the oracle's element-wise migration."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload
from oracle import oracle as O
from helpers import make_logical, shard_all
from gpu_helpers import upload, download


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _case(name):
    if name == "s5b":
        w = workload("s5b")
        return w["model"], w["old"], w["new"], w["seed"]
    base = dict(workload("s5b")["model"])                         # Llama style, untied, bf16 params + fp32 master / m / v
    if name == "d64_128":
        base.update(n_layers=8, hidden=96, n_q_heads=8, n_kv_heads=8, head_dim=12, ffn_hidden=192, vocab=1030, max_pos=0)
        return (base, dict(tp=4, pp=4, dp=4, dist_opt=1, vocab_divisor=8), dict(tp=8, pp=4, dp=4, dist_opt=1, vocab_divisor=8),
                0x64128)                                          # padded vocabulary 1056 -> 1088 rows
    if name == "p64_128":
        base.update(n_layers=8, hidden=128, n_q_heads=8, n_kv_heads=4, head_dim=16, ffn_hidden=320, vocab=1030, max_pos=0,
                    kinds=0b0011)
        return (base, dict(tp=2, pp=8, dp=4, dist_opt=0, vocab_divisor=8), dict(tp=4, pp=8, dp=4, dist_opt=0, vocab_divisor=8),
                0x128064)
    raise KeyError(name)


_MEMO = {}


def _oracle(name, dmap_key, dmap):
    """Oracle side of a case (layouts, payload, overlap, and the element-wise migration under `dmap`), memoised."""
    if name not in _MEMO:
        model, a, b, seed = _case(name)
        oo, on = O.Layout(model, a), O.Layout(model, b)
        src_np = shard_all(oo, make_logical(model, seed, "stamp", lts=oo.logical_tensors()))
        _MEMO[name] = dict(oo=oo, on=on, src=src_np, ov=O.overlap(oo, on), mig={})
    m = _MEMO[name]
    if dmap_key is not None and dmap_key not in m["mig"]:
        fill = np.zeros(m["on"].n_dev, np.int64)
        dst, T, _ = O.migrate(m["oo"], m["on"], np.asarray(dmap, np.int32), m["src"], fill_out=fill)
        m["mig"][dmap_key] = (dst, T, fill)
    return m


def _compare(on, dst, exp, tag):
    for key, e in exp.items():
        if e.shape[0]:
            got = download(dst[key], on.elem_bytes(key[1]))
            assert np.array_equal(got, e), (tag, key, int((got != e).sum()))


def _gpu_side(E, name):
    model, a, b, _ = _case(name)
    old, new = E.etc_layout_create(model, a), E.etc_layout_create(model, b)
    assert (old.n_dev + new.n_dev) * 4 > 384                      # beyond the parameter-block pointer tables
    return model, a, b, old, new


@pytest.mark.parametrize("name", ["s5b", "d64_128", "p64_128"])
@pytest.mark.parametrize("flags", [0, 1])
def test_many_devices_plan_and_migrate(E, name, flags):
    model, a, b, old, new = _gpu_side(E, name)
    m = _oracle(name, None, None)
    ov, need, hold = E.etc_cost_matrix(old, new)
    o_ov, o_need, o_hold = m["ov"]
    assert np.array_equal(ov.cpu().numpy(), o_ov) and np.array_equal(need.cpu().numpy(), o_need)
    assert np.array_equal(hold.cpu().numpy(), o_hold)
    dm, lb = E.etc_sketch(ov)
    assert int(lb.item()) == O.sketch_hungarian(o_ov)[1]
    dmap = dm.cpu().numpy()
    dst_o, T, fill = _oracle(name, "sketch", dmap)["mig"]["sketch"]
    plan = E.etc_plan_create(old, new, dm, flags)
    assert plan.validate() == 0
    st = plan.stats
    assert np.array_equal(plan.traffic(), T)
    assert st.fill_bytes == int(fill.sum()) and (name != "d64_128" or st.n_fills > 0)
    assert st.local_bytes + st.remote_bytes + st.fill_bytes == int(o_need.sum())
    src = upload(m["src"])
    for rep in range(2):                                          # the plan's pointer table is rewritten by every call
        dst = E.alloc_buffers(new, fill=0xA5 - rep)
        staging = torch.full((max(st.staging_bytes, 16),), 0xA5, dtype=torch.uint8, device="cuda")
        E.etc_migrate(plan, src, dst, staging)
        torch.cuda.synchronize()
        _compare(m["on"], dst, dst_o, (name, flags, rep))


@pytest.mark.parametrize("name", ["s5b", "d64_128"])
@pytest.mark.parametrize("cap", [2 * 65536, 1 << 34])
def test_many_devices_rounds(E, name, cap):
    model, a, b, old, new = _gpu_side(E, name)
    rng = np.random.default_rng(5)
    P = max(old.n_dev, new.n_dev)
    dmap = rng.permutation(P)[: new.n_dev].astype(np.int32)       # an arbitrary map: plenty of remote traffic
    m = _oracle(name, "perm5", dmap)
    dst_o, T, fill = m["mig"]["perm5"]
    for flags in (0, 1):
        plan = E.etc_plan_create(old, new, torch.from_numpy(dmap).cuda(), flags | E.ETC_KIND_MAJOR)
        rounds = E.etc_plan_set_rounds(plan, cap)
        assert plan.validate() == 0
        assert all(r.staging_bytes <= cap for r in rounds) and sum(r.staged_bytes for r in rounds) == plan.stats.staged_bytes
        staging = torch.full((max(max((r.staging_bytes for r in rounds), default=0), 16),), 0x5A, dtype=torch.uint8, device="cuda")
        out = {}
        for k in sorted({r.kind for r in rounds}):
            src_k = upload({key: v for key, v in m["src"].items() if key[1] == k})   # only kind k exists
            dst_k = {key: v for key, v in E.alloc_buffers(new, fill=0x5A).items() if key[1] == k}
            for i, r in enumerate(rounds):
                if r.kind == k:
                    staging.fill_(0x5A)
                    E.etc_migrate_round(plan, i, src_k, dst_k, staging)
            torch.cuda.synchronize()
            out.update(dst_k)
            del src_k
        assert np.array_equal(plan.traffic(), T)
        _compare(m["on"], out, dst_o, (name, cap, flags))


@pytest.mark.parametrize("name", ["p64_128", "d64_128"])
@pytest.mark.parametrize("flags", [0, 1, 4])
def test_many_devices_no_sync_plan(E, name, flags):
    """p64_128 is small enough for the plan to stay deferred (bound-sized grids, counts read on the device, the pointer
    table in device memory); d64_128's bound exceeds 32 768 work items, so ETC_NO_SYNC quietly takes the synchronising
    path — both must write the oracle's bytes."""
    model, a, b, old, new = _gpu_side(E, name)
    m = _oracle(name, None, None)
    dm, _ = E.etc_sketch(E.etc_cost_matrix(old, new)[0])
    dst_o, T, fill = _oracle(name, "sketch", dm.cpu().numpy())["mig"]["sketch"]
    src = upload(m["src"])
    staging = torch.full((max(E.etc_staging_bound(old, new, flags), 16),), 0x3C, dtype=torch.uint8, device="cuda")
    dst = E.alloc_buffers(new, fill=0x3C)
    plan = E.etc_plan_create(old, new, dm, flags | E.ETC_NO_SYNC)
    assert plan.deferred == (name == "p64_128")
    E.etc_migrate(plan, src, dst, staging)
    torch.cuda.synchronize()
    _compare(m["on"], dst, dst_o, (name, flags))
    assert np.array_equal(plan.traffic(), T) and plan.stats.fill_bytes == int(fill.sum())
    assert plan.validate() == 0
    for t in dst.values():                                        # resolved now: exact grids, same bytes
        t.fill_(0x77)
    E.etc_migrate(plan, src, dst, staging)
    torch.cuda.synchronize()
    _compare(m["on"], dst, dst_o, (name, flags, "resolved"))


@pytest.mark.parametrize("name", ["p64_128", "d64_128", "s5b"])
def test_many_devices_migrate_state_one_call(E, name):
    """etc_migrate_state with 32 < P <= 1024: inside the one call the sketch first tries the row-maximum
    certificate (stream-ordered scratch) and, where that cannot hold, runs the CTA Hungarian search.
      * s5b (512 -> 384): every new rank finds one of its maximal columns — the certificate decides;
      * the scale-out cases (64 -> 128): two new ranks want each old device — the search decides;
      * s5b with a mask that takes 32 of the devices the free sketch uses and offers 40 unused ones instead: the bound over the
        usable columns is out of reach (checked on the oracle's matrix below) — the search decides, under a mask."""
    model, a, b, old, new = _gpu_side(E, name)
    m = _oracle(name, None, None)
    o_ov = m["ov"][0]
    n_new, P = o_ov.shape
    src = upload(m["src"])
    staging = torch.full((max(E.etc_staging_bound(old, new), 16),), 0x3C, dtype=torch.uint8, device="cuda")
    dst = E.alloc_buffers(new, fill=0x3C)
    plan = E.etc_migrate_state(model, a, b, src, dst, staging)
    torch.cuda.synchronize()
    dmap = plan.device_map()
    ref_map, ref_obj = O.sketch_hungarian(o_ov)[:2]
    assert plan.stats.local_bytes == ref_obj
    assert (ref_obj == int(o_ov.max(axis=1).sum())) == (name == "s5b")            # which of the two sketch kernels decided
    dst_o = _oracle(name, "state", dmap)["mig"]["state"][0]
    _compare(m["on"], dst, dst_o, (name, "free"))
    if n_new == P:
        return                                                    # every device is needed: no mask leaves a feasible problem
    rng = np.random.default_rng(9)
    ref_map = np.asarray(ref_map)
    avail = np.zeros(P, bool); avail[ref_map] = True
    avail[rng.choice(ref_map, size=32, replace=False)] = False
    avail[np.setdiff1d(np.arange(P), ref_map)[:40]] = True
    ref_obj2 = O.sketch_hungarian(o_ov, avail)[1]
    assert 0 <= ref_obj2 < int(np.where(avail[None, :], o_ov, -1).max(axis=1).sum())   # no certificate under this mask
    for t in dst.values():
        t.fill_(0x3C)
    plan = E.etc_migrate_state(model, a, b, src, dst, staging, avail=torch.from_numpy(avail.astype(np.uint8)).cuda())
    torch.cuda.synchronize()
    dmap2 = plan.device_map()
    assert all(avail[p] for p in dmap2) and len(set(dmap2.tolist())) == len(dmap2)
    assert plan.stats.local_bytes == ref_obj2
    dst_o2 = _oracle(name, "state_masked", dmap2)["mig"]["state_masked"][0]
    _compare(m["on"], dst, dst_o2, (name, "masked"))
