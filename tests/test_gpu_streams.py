"""-m gpu: object lifetime across streams.  bench.py plans step i+1 on a side stream while the copy kernels of step i
still run on another stream and drops each plan / layout as soon as the next one exists.  The library frees its tables
with stream-ordered frees, so the free must be ordered after EVERY stream that still reads the tables (the legacy
default stream, a NULL cudaStream_t, included): otherwise the next plan reuses the memory under a running copy kernel.
The result must stay bit-identical to the oracle's element-wise migration."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload
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


@pytest.mark.parametrize("copy_on_default_stream", [True, False])
@pytest.mark.parametrize("name,flags", [("s3", 0), ("s5", 1)])
def test_pipelined_plans_dropped_early(E, name, flags, copy_on_default_stream):
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    src = upload(src_np)
    lay_new = E.etc_layout_create(model, w["new"])
    dst = E.alloc_buffers(lay_new, fill=0x3C)
    plan_stream = torch.cuda.Stream(priority=-1)
    copy_stream = torch.cuda.default_stream() if copy_on_default_stream else torch.cuda.Stream()
    # a big dummy copy keeps the copy stream busy so that the planning of later steps runs far ahead of it
    big_a = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
    big_b = torch.empty_like(big_a)
    staging = None
    dmap = None
    for it in range(12):
        with torch.cuda.stream(plan_stream):
            lo, ln = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
            ov, _, _ = E.etc_cost_matrix(lo, ln, stream=plan_stream)
            dm, _ = E.etc_sketch(ov, stream=plan_stream)
            plan = E.etc_plan_create(lo, ln, dm, flags, stream=plan_stream)
            done = torch.cuda.Event()
            done.record(plan_stream)
        if staging is None:
            staging = torch.empty(max(plan.stats.staging_bytes, 16), dtype=torch.uint8, device="cuda")
            dmap = dm.cpu().numpy().copy()
        assert plan.stats.staging_bytes <= staging.numel()
        with torch.cuda.stream(copy_stream):
            for _ in range(3):
                big_b.copy_(big_a, non_blocking=True)
            copy_stream.wait_event(done)
            E.etc_migrate(plan, src, dst, staging, stream=copy_stream)
        del plan, lo, ln            # dropped while the copy stream is still far behind
    torch.cuda.synchronize()
    exp, _, _ = oracle_migrate(oo, on, dmap, src_np)
    for key, e in exp.items():
        if e.shape[0]:
            assert np.array_equal(download(dst[key], on.elem_bytes(key[1])), e), key


@pytest.mark.parametrize("name,flags", [("c1", 0), ("s4odd", 1), ("s5", 0)])
def test_migrate_is_cuda_graph_capturable(E, name, flags):
    """include/etc.h: etc_migrate does no allocation and no host synchronisation (its pointer tables travel as kernel
    parameters, not as copies from pageable memory), so it can be captured into a CUDA graph and replayed: the replay
    on fresh payloads must still equal the oracle's element-wise migration."""
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    payloads = [sharded_payload(oo, w["seed"] + i, "stamp" if i == 0 else "salted") for i in range(3)]
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    dm, _ = E.etc_sketch(E.etc_cost_matrix(old, new)[0])
    plan = E.etc_plan_create(old, new, dm, flags)
    src = upload(payloads[0])
    dst = E.alloc_buffers(new, fill=0x3C)
    staging = torch.empty(max(plan.stats.staging_bytes, 16), dtype=torch.uint8, device="cuda")
    E.etc_migrate(plan, src, dst, staging)                         # warm-up: kernel attributes are set outside capture
    torch.cuda.synchronize()
    launches0 = E.kernel_launches()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        E.etc_migrate(plan, src, dst, staging)
    per_call = E.kernel_launches() - launches0
    assert 1 <= per_call <= 4
    dm_h = dm.cpu().numpy()
    for i in (1, 2):
        for key, a in payloads[i].items():
            if a.shape[0]:
                src[key].copy_(torch.from_numpy(a.view(np.uint8).copy()))
        for t in dst.values():
            t.fill_(0x3C)
        graph.replay()
        torch.cuda.synchronize()
        exp, _, _ = oracle_migrate(oo, on, dm_h, payloads[i])
        for key, e in exp.items():
            if e.shape[0]:
                assert np.array_equal(download(dst[key], e.itemsize), e), (i, key)


@pytest.mark.parametrize("name,flags", [("s3", 0), ("s4", 1)])
def test_plan_used_on_another_stream_without_a_manual_wait(E, name, flags):
    """include/etc.h etc_plan_create: the slice and chunk tables are written by kernels enqueued AFTER the call's one host
    synchronisation, so the plan is complete in stream order only.  A call that reads it on another stream must order
    itself after those kernels (the library records an event at the end of etc_plan_create and waits for it).  Here the
    planning stream is held back by a long dummy copy enqueued before the plan's table kernels could run... the
    migration on a second stream, with NO wait_event by the caller, must still equal the oracle; so must
    etc_plan_validate and etc_plan_set_rounds + etc_migrate_round on a third stream."""
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    src = upload(src_np)
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    dm, _ = E.etc_sketch(E.etc_cost_matrix(old, new)[0])
    torch.cuda.synchronize()
    dmap = dm.cpu().numpy().copy()
    exp, _, _ = oracle_migrate(oo, on, dmap, src_np)
    big_a = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
    big_b = torch.empty_like(big_a)
    s_plan, s_copy, s_rounds = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    for mode in ("migrate", "rounds"):
        dst = E.alloc_buffers(new, fill=0x3C)
        torch.cuda.synchronize()
        with torch.cuda.stream(s_plan):
            # etc_plan_create synchronises s_plan once (sizes), then enqueues the table kernels behind these copies: a
            # second thread keeps the stream fed while the call waits
            import threading
            stop = threading.Event()

            def feed():
                with torch.cuda.stream(s_plan):
                    while not stop.is_set():
                        for _ in range(4):
                            big_b.copy_(big_a, non_blocking=True)
                        stop.wait(0.0005)
            th = threading.Thread(target=feed)
            th.start()
            try:
                plan = E.etc_plan_create(old, new, dm, flags | (E.ETC_KIND_MAJOR if mode == "rounds" else 0), stream=s_plan)
            finally:
                stop.set(); th.join()
        staging = torch.empty(max(plan.stats.staging_bytes, 16), dtype=torch.uint8, device="cuda")
        if mode == "migrate":
            E.etc_migrate(plan, src, dst, staging, stream=s_copy)          # no wait_event here
            assert plan.validate(stream=s_rounds) == 0
        else:
            rounds = E.etc_plan_set_rounds(plan, max(2 * 65536, plan.stats.staging_bytes // 3 + 65536), stream=s_rounds)
            for i in range(len(rounds)):
                E.etc_migrate_round(plan, i, src, dst, staging, stream=s_copy)
        torch.cuda.synchronize()
        for key, e in exp.items():
            if e.shape[0]:
                assert np.array_equal(download(dst[key], on.elem_bytes(key[1])), e), (mode, key)
        del plan


@pytest.mark.parametrize("name,flags", [("s3", 0), ("s5", 1), ("s4odd", 0)])
def test_one_plan_two_host_threads(E, name, flags):
    """include/etc.h "Concurrency": a plan is immutable and may be used by several etc_migrate* calls at once, from different
    host threads, on different streams with different buffer sets.  Two threads start together (a
    barrier) on a FRESH plan — so the first-use set-up inside the library (kernel attributes, the plan's ready event) is hit
    from both — and each migrates its own payload 8 times; an ETC_NO_SYNC plan is used the same way, so that both threads
    also race to resolve its device-side counts.  Every result must equal the oracle's element-wise migration."""
    import threading
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    payloads = [sharded_payload(oo, w["seed"] + 10 + i, "stamp" if i == 0 else "salted") for i in range(2)]
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    dm, _ = E.etc_sketch(E.etc_cost_matrix(old, new)[0])
    dm_h = dm.cpu().numpy()
    exp = [oracle_migrate(oo, on, dm_h, p)[0] for p in payloads]
    srcs = [upload(p) for p in payloads]
    bound = max(E.etc_staging_bound(old, new, flags), 16)
    for plan_flags in (flags, flags | E.ETC_NO_SYNC):
        plan = E.etc_plan_create(old, new, dm, plan_flags)
        dsts = [E.alloc_buffers(new, fill=0x3C) for _ in range(2)]
        stagings = [torch.full((bound,), 0x3C, dtype=torch.uint8, device="cuda") for _ in range(2)]
        streams = [torch.cuda.Stream() for _ in range(2)]
        torch.cuda.synchronize()
        gate = threading.Barrier(2)
        errors = []

        def worker(i):
            try:
                torch.cuda.set_device(dsts[i][next(iter(dsts[i]))].device)
                gate.wait()
                for rep in range(8):
                    E.etc_migrate(plan, srcs[i], dsts[i], stagings[i], stream=streams[i])
                    if rep == 3:
                        assert plan.stats.n_old == old.n_dev       # resolves a deferred plan from both threads
                streams[i].synchronize()
            except Exception as ex:                                # surfaced below: an assert in a thread is otherwise lost
                errors.append((i, repr(ex)))

        threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        torch.cuda.synchronize()
        assert not errors, errors
        for i in range(2):
            for key, e in exp[i].items():
                if e.shape[0]:
                    assert np.array_equal(download(dsts[i][key], on.elem_bytes(key[1])), e), (plan_flags, i, key)
