"""-m gpu tests of the address-ordered launch lists (csrc/plan_order.cu; PAPER.md:197 pack / unpack).

A plan keeps its copy work items ("chunks") a second time in the order the launches walk them: launch 1 (pack + local)
by source address, launch 2 (unpack) by destination address.  Checked here, through the C ABI:
  * the ordered lists are PERMUTATIONS of the plan's chunk lists (record by record), and are in address order;
  * the chunks of a list cover every destination byte exactly once (so a permutation bug cannot hide behind a duplicate);
  * migration through the ordered lists == migration in list order (ETC_NO_REORDER) == the element-wise oracle, from
    poisoned destinations, whole plans and rounds of bounded staging;
  * a plan that keeps no ordered lists says so.
"""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload
from oracle import oracle as O
from helpers import sharded_payload, oracle_migrate, random_variant_case
from gpu_helpers import upload, download, run_gpu_migration


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


FIELDS = ("src_off", "dst_off", "stg_off", "src_stride", "dst_stride", "row_bytes", "nrows", "src_buf", "dst_buf", "vec")


def _records(arr, staged=None):
    """chunk records as sortable rows (the `staged` column taken from the argument for the plan's own lists)"""
    cols = [arr[f].astype(np.int64) for f in FIELDS]
    cols.append(arr["staged"].astype(np.int64) if staged is None else np.full(arr.shape[0], staged, np.int64))
    m = np.stack(cols, axis=1) if arr.shape[0] else np.zeros((0, len(FIELDS) + 1), np.int64)
    return m[np.lexsort(m.T[::-1])]


def _in_address_order(buf, off):
    """non-decreasing buffer index, and inside a buffer non-decreasing 64 KB block (include/etc.h, etc_plan_get_chunks)"""
    key = buf.astype(np.int64) * (1 << 40) + (off.astype(np.int64) >> 16)
    return bool(np.all(np.diff(key) >= 0))


def _plan(E, w, flags, device_map=None):
    old, new = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    if device_map is None:
        ov, _, _ = E.etc_cost_matrix(old, new)
        dm, _ = E.etc_sketch(ov)
    else:
        dm = torch.tensor(np.asarray(device_map, np.int32)).cuda()
    return old, new, E.etc_plan_create(old, new, dm, flags)


@pytest.mark.parametrize("name", ["c1", "s2", "s3", "s4", "s4odd", "s5", "sx64", "sx64r", "sxodd"])
@pytest.mark.parametrize("flags", [0, 1, 2, 4])
def test_ordered_lists_are_sorted_permutations(E, name, flags):
    w = workload(name)
    old, new, plan = _plan(E, w, flags)
    _check_lists(plan, new)


@pytest.mark.parametrize("name", ["s3", "s5"])
@pytest.mark.parametrize("flags", [0, 1])
def test_no_sync_plans_keep_ordered_lists_when_the_state_exceeds_l2(E, name, flags):
    """A bound-sized ETC_NO_SYNC plan sorts with bound-sized grids and device-side counts (states of 128 MB and more)."""
    w = workload(name)
    old, new, plan = _plan(E, w, flags | E.ETC_NO_SYNC)
    assert new.total_bytes() >= 128 << 20
    _check_lists(plan, new)
    # and the migration through them == oracle
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    src, dst = upload(src_np), E.alloc_buffers(new, fill=0x4D)
    staging = torch.full((max(E.etc_staging_bound(old, new, flags), 16),), 0x4D, dtype=torch.uint8, device="cuda")
    E.etc_migrate(plan, src, dst, staging)
    torch.cuda.synchronize()
    exp, T, _ = oracle_migrate(oo, on, plan.device_map(), src_np)
    assert np.array_equal(plan.traffic(), T)
    for (n, k), e in exp.items():
        if e.shape[0]:
            assert np.array_equal(download(dst[(n, k)], e.itemsize), e), (n, k)


def _check_lists(plan, new):
    st = plan.stats
    a, b = plan.chunks(0), plan.chunks(1)
    l1, l2 = plan.chunks(2), plan.chunks(3)
    assert a.shape[0] == st.n_chunks_staged and b.shape[0] == st.n_chunks_local
    assert l1.shape[0] == a.shape[0] + b.shape[0] and l2.shape[0] == a.shape[0]
    assert not a["staged"].any() and not b["staged"].any() and not l2["staged"].any()
    both = np.concatenate([_records(a, 1), _records(b, 0)])
    both = both[np.lexsort(both.T[::-1])]
    assert np.array_equal(_records(l1), both)                       # launch 1 holds exactly the plan's chunks
    assert np.array_equal(_records(l2, 1), _records(a, 1))          # launch 2 exactly the staged ones
    assert _in_address_order(l1["src_buf"], l1["src_off"])
    assert _in_address_order(l2["dst_buf"], l2["dst_off"])
    assert plan.validate() == 0
    # every destination byte once: local chunks of launch 1 + all chunks of launch 2
    cover = {}
    for n in range(new.n_dev):
        for k in range(4):
            cover[n * 4 + k] = np.zeros(new.buffer_bytes(n, k), np.uint8)
    from numpy.lib.stride_tricks import as_strided
    for c in list(l1[l1["staged"] == 0]) + list(l2):
        buf, nrows, rb, a0 = cover[int(c["dst_buf"])], int(c["nrows"]), int(c["row_bytes"]), int(c["dst_off"])
        pitch = int(c["dst_stride"]) if nrows > 1 else rb
        as_strided(buf[a0:], shape=(nrows, rb), strides=(pitch, 1))[...] += 1
    for key, c in cover.items():
        assert np.all(c == 1), key


@pytest.mark.parametrize("name", ["s3", "s4", "sx64", "c1"])
def test_ordered_lists_are_deterministic(E, name):
    """The order inside an address bin is fixed by a per-bin sort: two plans of the same reconfiguration keep identical
    launch lists, record for record (the histogram's atomics alone would leave it to chance)."""
    w = workload(name)
    lists = []
    for _ in range(3):
        old, new, plan = _plan(E, w, 0)
        lists.append((plan.chunks(2).copy(), plan.chunks(3).copy()))
        assert plan.validate() == 0
    for l1, l2 in lists[1:]:
        assert np.array_equal(l1, lists[0][0]) and np.array_equal(l2, lists[0][1])


def test_plans_without_ordered_lists_say_so(E):
    w = workload("s2")
    for flags in (E.ETC_NO_REORDER, E.ETC_NO_SYNC):
        old, new, plan = _plan(E, w, flags)
        assert plan.chunks(0).shape[0] + plan.chunks(1).shape[0] > 0
        for which in (2, 3):
            with pytest.raises(E.EtcError):
                plan.chunks(which)
        assert plan.validate() == 0


def _migrate(E, w, src_np, flags, device_map, poison):
    g = run_gpu_migration(w["model"], w["old"], w["new"], src_np, device_map=device_map, flags=flags, poison=poison)
    return g


@pytest.mark.parametrize("name", ["s2", "s3", "s4", "s4odd", "s5", "sx64", "sx64r", "sxodd"])
def test_ordered_and_list_order_launches_agree_with_the_oracle(E, name):
    w = workload(name)
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    src = sharded_payload(oo, w["seed"], "stamp")
    for flags in (0, 1):
        g1 = _migrate(E, w, src, flags, None, 0xA5)
        dm = g1["device_map"]
        g0 = _migrate(E, w, src, flags | E.ETC_NO_REORDER, dm, 0x3C)
        exp, T, _ = oracle_migrate(oo, on, dm, src)
        assert np.array_equal(g1["plan"].traffic(), T) and np.array_equal(g0["plan"].traffic(), T)
        for key, e in exp.items():
            assert np.array_equal(g1["dst"][key], e), ("ordered", key)
            assert np.array_equal(g0["dst"][key], e), ("list order", key)


def test_random_variants_ordered_vs_list_order(E):
    rng = np.random.default_rng(2607)
    ran = 0
    for t in range(40):
        model, a, b = random_variant_case(rng)
        oo, on = O.Layout(model, a), O.Layout(model, b)
        w = dict(model=model, old=a, new=b)
        src = sharded_payload(oo, 700 + t, "stamp", padded_lts=True)
        nn, no = on.n_dev, oo.n_dev
        dm = None if t % 2 else rng.permutation(max(nn, no))[:nn].astype(np.int32)
        flags = int(rng.choice([0, 1, 2, 3, 4, 6]))
        g1 = _migrate(E, w, src, flags, dm, 0xA5)
        g0 = _migrate(E, w, src, flags | E.ETC_NO_REORDER, g1["device_map"], 0x3C)
        exp, T, _ = oracle_migrate(oo, on, g1["device_map"], src)
        for key, e in exp.items():
            assert np.array_equal(g1["dst"][key], e), (t, "ordered", key)
            assert np.array_equal(g0["dst"][key], e), (t, "list order", key)
        ran += 1
    assert ran == 40


@pytest.mark.parametrize("name", ["s4", "sx64"])
@pytest.mark.parametrize("cap", [1 << 17, 1 << 20])
def test_rounds_walk_ordered_lists(E, name, cap):
    """Rounds of bounded staging use per-round ordered lists (checked by etc_plan_validate: bounds + permutation) and
    write what the oracle writes; with ETC_NO_REORDER they walk the chunk ranges in list order — same bytes."""
    w = workload(name)
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    outs = []
    for extra in (0, E.ETC_NO_REORDER):
        old, new, plan = _plan(E, w, E.ETC_ALL_STAGED | E.ETC_KIND_MAJOR | extra)
        rounds = E.etc_plan_set_rounds(plan, cap)
        assert plan.validate() == 0
        src = upload(src_np)
        dst = E.alloc_buffers(new, fill=0x77)
        staging = torch.full((max(max((r.staging_bytes for r in rounds), default=0), 16),), 0x77, dtype=torch.uint8, device="cuda")
        for i, r in enumerate(rounds):
            staging.fill_(0x77)
            E.etc_migrate_round(plan, i, src, dst, staging)
        torch.cuda.synchronize()
        outs.append((plan, {k: v.cpu().numpy() for k, v in dst.items()}))
    (p1, d1), (p0, d0) = outs
    for key in d1:
        assert np.array_equal(d1[key], d0[key]), key
    exp, _, _ = oracle_migrate(oo, on, p1.device_map(), src_np)
    for (n, k), e in exp.items():
        if e.shape[0]:
            assert np.array_equal(d1[(n, k)].view(e.dtype), e), (n, k)


def test_ordered_lists_of_the_512_to_384_device_layout(E):
    """c5b (3.95 TB of virtual state, metadata only): 45 M chunks, more than 4 M 64 KB blocks, so the sort uses coarser
    address bins (1 MB here) — the lists must still be bounds-checked permutations in (coarser) address order."""
    w = workload("c5b")
    old, new, plan = _plan(E, w, E.ETC_ALL_STAGED)
    st = plan.stats
    assert st.n_chunks_staged > 40_000_000 and st.remote_bytes == 0 and st.local_bytes == new.total_bytes()
    assert plan.validate() == 0                       # bounds + permutation checksums of both ordered lists
    assert old.total_bytes() >> 16 > 1 << 22           # more 64 KB blocks than the sort has bins: coarser bins
    shift = 23                                        # 16 MB blocks: coarser than any bin size the sort may pick here
    l1 = plan.chunks(2)
    assert l1.shape[0] == st.n_chunks_staged and bool(l1["staged"].all())
    key = l1["src_buf"].astype(np.int64) * (1 << 44) + (l1["src_off"].astype(np.int64) >> (shift + 1))
    assert np.all(np.diff(key) >= 0)
    del l1, key
    l2 = plan.chunks(3)
    key = l2["dst_buf"].astype(np.int64) * (1 << 44) + (l2["dst_off"].astype(np.int64) >> (shift + 1))
    assert np.all(np.diff(key) >= 0)
