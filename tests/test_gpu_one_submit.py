"""-m gpu: the path without host synchronisation (PAPER.md:368 — the metadata steps are "almost
negligible", so a small reconfiguration should cost its kernels, not host round trips).
  * ETC_NO_SYNC plans: tables sized from host-side bounds, counts on the device, bound-sized copy grids — must write exactly
    what the element-wise oracle writes, report the same statistics as a plan made the synchronising way, and detect bad
    maps on the device;
  * etc_migrate_state: (a1)-(a6) in ONE C-ABI call;
  * the whole of (a2)-(a6) captured into ONE CUDA graph and replayed on fresh payloads."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload
from oracle import oracle as O
from helpers import sharded_payload, oracle_migrate, oracle_overlap, random_variant_case, make_logical, shard_all
from gpu_helpers import upload, download


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _compare(on, dst, exp, tag):
    for key, e in exp.items():
        if e.shape[0]:
            assert np.array_equal(download(dst[key], on.elem_bytes(key[1])), e), (tag, key)


@pytest.mark.parametrize("name", ["c1", "s2", "s2odd", "s3", "s4", "s4odd", "s5"])
@pytest.mark.parametrize("flags", [0, 1, 4])
def test_no_sync_plan_vs_oracle_and_vs_synchronising_plan(E, name, flags):
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    src = upload(src_np)
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    dm, _ = E.etc_sketch(E.etc_cost_matrix(old, new)[0])
    bound = E.etc_staging_bound(old, new, flags)
    ref = E.etc_plan_create(old, new, dm, flags)
    assert ref.stats.staging_bytes <= bound
    staging = torch.full((max(bound, 16),), 0x3C, dtype=torch.uint8, device="cuda")
    dst = E.alloc_buffers(new, fill=0x3C)
    launches0 = E.kernel_launches()
    plan = E.etc_plan_create(old, new, dm, flags | E.ETC_NO_SYNC)
    E.etc_migrate(plan, src, dst, staging)                    # enqueued before any count has reached the host
    assert plan._stats is None
    torch.cuda.synchronize()
    # count, scan, fill, two copy launches, table uploads; + base-table upload and 4 sort launches when the state is big
    # enough for the plan to keep address-ordered launch lists (csrc/plan_order.cu)
    assert E.kernel_launches() - launches0 <= (14 if new.total_bytes() >= 128 << 20 else 9)
    exp, T, _ = oracle_migrate(oo, on, dm.cpu().numpy(), src_np)
    _compare(on, dst, exp, name)
    a, b = plan.stats, ref.stats
    for f in ("staging_bytes", "local_bytes", "remote_bytes", "staged_bytes", "n_slices_local", "n_slices_staged",
              "n_chunks_local", "n_chunks_staged", "fill_bytes", "n_fills", "flags"):
        assert getattr(a, f) == getattr(b, f), f
    assert np.array_equal(plan.traffic(), T)
    assert plan.validate() == 0
    assert np.array_equal(plan.device_map(), dm.cpu().numpy())
    # once resolved, the plan migrates with exact grids; and it can be cut into rounds like any other kind-major plan
    for t in dst.values():
        t.fill_(0x77)
    E.etc_migrate(plan, src, dst, staging)
    torch.cuda.synchronize()
    _compare(on, dst, exp, name + " resolved")


def test_no_sync_plan_detects_bad_maps_on_the_device(E):
    w = workload("s3")
    old, new = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    src = E.alloc_buffers(old, fill=1)
    dst = E.alloc_buffers(new, fill=0x3C)
    staging = torch.empty(E.etc_staging_bound(old, new), dtype=torch.uint8, device="cuda")
    for bad in ([0] * new.n_dev, list(range(new.n_dev - 1)) + [99], [-1] * new.n_dev):
        dm = torch.tensor(bad, dtype=torch.int32, device="cuda")          # a DEVICE map: the host cannot look at it
        plan = E.etc_plan_create(old, new, dm, E.ETC_NO_SYNC)
        E.etc_migrate(plan, src, dst, staging)
        torch.cuda.synchronize()
        for t in dst.values():
            assert bool((t == 0x3C).all())                                # nothing was copied
        with pytest.raises(E.EtcError) as e:
            plan.stats
        assert e.value.code == -4                                         # ETC_ERR_BAD_MAP


def test_unusable_no_sync_plan_is_reported_by_every_query_and_writes_nothing(E):
    """include/etc.h: a device-detected error of an ETC_NO_SYNC plan (here a map that is not injective) comes back from
    EVERY call that needs the plan's counts on the host — not only etc_plan_get_stats — and such a plan writes nothing,
    the zero-fill of a grown padded vocabulary (reading A31) included.  Raw C-ABI calls: the Python wrappers read .stats
    first and would hide which entry point reported the error."""
    import ctypes as C
    from test_vocab_padding_pins import _model, _cfg
    model, a, b = _model(), _cfg(1), _cfg(2)                      # vocab 5 padded to 6 -> 8 rows: the new layout has fill rows
    old, new = E.etc_layout_create(model, a), E.etc_layout_create(model, b)
    src = E.alloc_buffers(old, fill=1)
    staging = torch.empty(max(E.etc_staging_bound(old, new, E.ETC_KIND_MAJOR), 16), dtype=torch.uint8, device="cuda")
    good = E.etc_plan_create(old, new, torch.arange(new.n_dev, dtype=torch.int32, device="cuda"), E.ETC_NO_SYNC | E.ETC_KIND_MAJOR)
    assert good.stats.n_fills > 0                                 # the case does have bytes with no source
    L = E.lib()
    for order in range(5):
        dst = E.alloc_buffers(new, fill=0x3C)
        dm = torch.zeros(new.n_dev, dtype=torch.int32, device="cuda")     # both new ranks on device 0
        plan = E.etc_plan_create(old, new, dm, E.ETC_NO_SYNC | E.ETC_KIND_MAJOR)
        E.etc_migrate(plan, src, dst, staging)
        torch.cuda.synchronize()
        for t in dst.values():
            assert bool((t == 0x3C).all())                        # not even the padded vocabulary rows were zeroed
        n_bad, n_rounds = C.c_int64(-9), C.c_int32(-9)
        T = np.full((2, 2), -9, np.int64)
        rec = np.zeros(4096, np.uint8)
        calls = [lambda: L.etc_plan_validate(plan.h, C.byref(n_bad), 0),
                 lambda: L.etc_plan_set_rounds(plan.h, 1 << 20, C.byref(n_rounds), 0),
                 lambda: L.etc_plan_get_traffic(plan.h, T.ctypes.data),
                 lambda: L.etc_plan_get_slices(plan.h, 0, rec.ctypes.data),
                 lambda: L.etc_plan_get_fills(plan.h, rec.ctypes.data)]
        calls = calls[order:] + calls[:order]                     # each of them is once the FIRST query of a fresh plan
        for call in calls:
            assert call() == -4                                   # ETC_ERR_BAD_MAP
        assert n_bad.value == -9 and n_rounds.value == -9 and (T == -9).all() and not rec.any()   # outputs untouched


def test_no_sync_plan_with_variants_failures_and_fills(E):
    """Random reconfigurations drawing on every layout variant (incl. grown padded vocabularies -> zero-fill list with a
    device-side count) and failure masks through ETC_NO_SYNC plans."""
    rng = np.random.default_rng(77)
    ran = fills = 0
    for t in range(40):
        model, a, b = random_variant_case(rng)
        oo, on = O.Layout(model, a), O.Layout(model, b)
        src_np = shard_all(oo, make_logical(model, 900 + t, "stamp", lts=oo.logical_tensors()))
        old, new = E.etc_layout_create(model, a), E.etc_layout_create(model, b)
        P = max(old.n_dev, new.n_dev)
        dmap = rng.permutation(P)[: new.n_dev].astype(np.int32)
        flags = int(rng.choice([0, 1, 4]))
        fill = np.zeros(on.n_dev, np.int64)
        exp, T, _ = O.migrate(oo, on, dmap, src_np, fill_out=fill)
        src = upload(src_np)
        dst = E.alloc_buffers(new, fill=0x3C)
        staging = torch.full((max(E.etc_staging_bound(old, new, flags), 16),), 0x3C, dtype=torch.uint8, device="cuda")
        plan = E.etc_plan_create(old, new, torch.from_numpy(dmap).cuda(), flags | E.ETC_NO_SYNC)
        E.etc_migrate(plan, src, dst, staging)
        torch.cuda.synchronize()
        _compare(on, dst, exp, t)
        assert plan.stats.fill_bytes == int(fill.sum())
        assert np.array_equal(plan.traffic(), T)
        fills += plan.stats.n_fills > 0
        ran += 1
    assert ran == 40 and fills >= 3


@pytest.mark.parametrize("name,flags", [("c1", 0), ("s2", 0), ("s3", 1), ("s4", 0), ("s5", 0), ("s4odd", 4)])
def test_migrate_state_is_one_call(E, name, flags):
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    src = upload(src_np)
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    staging = torch.full((max(E.etc_staging_bound(old, new, flags), 16),), 0x3C, dtype=torch.uint8, device="cuda")
    dst = E.alloc_buffers(new, fill=0x3C)
    call = E.MigrateState(model, w["old"], w["new"], src, dst, staging, flags)
    plan = call(want_plan=True)
    torch.cuda.synchronize()
    dmap = plan.device_map()
    o_ov, _, _ = oracle_overlap(oo, on)
    assert plan.stats.local_bytes == (O.sketch_bruteforce(o_ov)[1] if o_ov.shape[1] <= 8 else O.sketch_hungarian(o_ov)[1])
    exp, T, _ = oracle_migrate(oo, on, dmap, src_np)
    _compare(on, dst, exp, name)
    assert np.array_equal(plan.traffic(), T)
    # fire and forget (no plan returned), several in a row on fresh poison: still exact
    for i in range(3):
        for t in dst.values():
            t.fill_(0x11 * (i + 1))
        assert call() is None
    torch.cuda.synchronize()
    _compare(on, dst, exp, name + " repeat")
    # staging smaller than the bound is refused before anything is enqueued
    if flags != 4 and staging.numel() > 4096:
        with pytest.raises(E.EtcError) as e:
            E.MigrateState(model, w["old"], w["new"], src, dst, staging[: staging.numel() // 2], flags)()
        assert e.value.code == -5


def test_migrate_state_with_availability_mask(E):
    w = workload("s3")                                   # 16 -> 12 devices; forbid the devices the free sketch would keep
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    src = upload(src_np)
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    staging = torch.empty(E.etc_staging_bound(old, new), dtype=torch.uint8, device="cuda")
    dst = E.alloc_buffers(new, fill=0x3C)
    avail = np.ones(16, np.uint8); avail[[12, 13, 14, 15]] = 0
    plan = E.etc_migrate_state(model, w["old"], w["new"], src, dst, staging, avail=torch.from_numpy(avail).cuda())
    torch.cuda.synchronize()
    dmap = plan.device_map()
    assert set(dmap.tolist()).isdisjoint({12, 13, 14, 15})
    o_ov, _, _ = oracle_overlap(oo, on)
    assert plan.stats.local_bytes == O.sketch_hungarian(o_ov, avail)[1]
    exp, _, _ = oracle_migrate(oo, on, dmap, src_np)
    _compare(on, dst, exp, "avail")
    # an infeasible mask: the sketch writes -1, the plan sees a bad map on the device and copies nothing
    for t in dst.values():
        t.fill_(0x3C)
    avail[:] = 0; avail[:5] = 1
    plan = E.etc_migrate_state(model, w["old"], w["new"], src, dst, staging, avail=torch.from_numpy(avail).cuda())
    torch.cuda.synchronize()
    assert all(bool((t == 0x3C).all()) for t in dst.values())
    with pytest.raises(E.EtcError) as e:
        plan.stats
    assert e.value.code == -4


@pytest.mark.parametrize("name,flags", [("c1", 0), ("s3", 0), ("s5", 1)])
def test_whole_path_in_one_cuda_graph(E, name, flags):
    """(a2) cost matrix, (a3) sketch, (a4) ETC_NO_SYNC plan, (a5, a6) copy launches and the plan's stream-ordered release
    captured into ONE CUDA graph (no allocation outside the graph's own nodes, no host synchronisation), replayed on fresh
    payloads: bit-identical to the oracle with the map the captured sketch chose."""
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    payloads = [sharded_payload(oo, w["seed"] + i, "stamp" if i == 0 else "salted") for i in range(3)]
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    src = upload(payloads[0])
    dst = E.alloc_buffers(new, fill=0x3C)
    staging = torch.empty(max(E.etc_staging_bound(old, new, flags), 16), dtype=torch.uint8, device="cuda")
    P = max(old.n_dev, new.n_dev)
    out_cost = (torch.empty((new.n_dev, P), dtype=torch.int64, device="cuda"), torch.empty(new.n_dev, dtype=torch.int64, device="cuda"),
                torch.empty(P, dtype=torch.int64, device="cuda"))
    out_sk = (torch.empty(new.n_dev, dtype=torch.int32, device="cuda"), torch.empty(1, dtype=torch.int64, device="cuda"))

    def whole_path():
        ov, _, _ = E.etc_cost_matrix(old, new, out=out_cost)
        dm, _ = E.etc_sketch(ov, out=out_sk)
        plan = E.etc_plan_create(old, new, dm, flags | E.ETC_NO_SYNC)
        E.etc_migrate(plan, src, dst, staging)
        del plan                                          # released in stream order, inside the capture
    whole_path()                                          # warm-up: kernel attributes, memory pool
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        whole_path()
    dm_h = None
    for i in (1, 2):
        for key, a in payloads[i].items():
            if a.shape[0]:
                src[key].copy_(torch.from_numpy(a.view(np.uint8).copy()))
        for t in dst.values():
            t.fill_(0x3C)
        out_sk[0].fill_(-7)
        graph.replay()
        torch.cuda.synchronize()
        dm_h = out_sk[0].cpu().numpy()
        exp, _, _ = oracle_migrate(oo, on, dm_h, payloads[i])
        _compare(on, dst, exp, (name, i))


def test_many_interleaved_one_call_migrations(E):
    """Back-to-back etc_migrate_state calls of reconfigurations of different sizes on two streams, with no host
    synchronisation in between: the layout upload slabs are reused while earlier uploads may still be in flight, plans and
    layouts are released in stream order while their kernels are queued.  Every result must still equal the oracle."""
    cases = []
    for name, flags in (("c1", 0), ("s4", 0), ("s2odd", 1), ("s3", 4), ("sx64", 0)):
        w = workload(name)
        model = w["model"]
        oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
        src_np = sharded_payload(oo, w["seed"], "stamp")
        old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
        src, dst = upload(src_np), E.alloc_buffers(new, fill=0x3C)
        staging = torch.empty(max(E.etc_staging_bound(old, new, flags), 16), dtype=torch.uint8, device="cuda")
        cases.append(dict(name=name, oo=oo, on=on, src_np=src_np, dst=dst,
                          call=E.MigrateState(model, w["old"], w["new"], src, dst, staging, flags)))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    plans = {}
    for it in range(40):
        for j, c in enumerate(cases):
            st = streams[j % 2]                          # a case always runs on the same stream (its buffers are reused)
            last = it == 39
            p = c["call"](stream=st, want_plan=last)
            if last:
                plans[c["name"]] = p
    torch.cuda.synchronize()
    for c in cases:
        dmap = plans[c["name"]].device_map()
        exp, T, _ = oracle_migrate(c["oo"], c["on"], dmap, c["src_np"])
        _compare(c["on"], c["dst"], exp, c["name"])
        assert np.array_equal(plans[c["name"]].traffic(), T)
