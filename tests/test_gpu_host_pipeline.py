"""-m gpu parity of the host-resident pipeline (bench.py's e2e leg) and of the chunked, eagerly-releasing device
migration (f2) against the element-wise oracle."""
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


def _pinned(np_bufs):
    out = {}
    for key, a in np_bufs.items():
        if a.shape[0]:
            t = torch.empty(a.nbytes, dtype=torch.uint8, pin_memory=True)
            t.numpy()[:] = a.view(np.uint8)
            out[key] = t
    return out


@pytest.mark.parametrize("name", ["c1", "s3", "s4", "s5"])
@pytest.mark.parametrize("cap", [2 * 65536, 1 << 24])
def test_host_migration_vs_oracle(E, name, cap):
    from paper_2607_04749_b200.host_pipeline import HostMigration
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    payloads = [sharded_payload(oo, w["seed"] + i, "stamp" if i == 0 else "salted") for i in range(2)]
    h_src = _pinned(payloads[0])
    h_dst = {(n, k): torch.full((on.buffer_elems(n, k) * on.elem_bytes(k),), 0x77, dtype=torch.uint8).pin_memory()
             for n in range(on.n_dev) for k in on.kinds() if on.buffer_elems(n, k)}
    hm = HostMigration(model, w["old"], w["new"], h_src, h_dst, max_staging_bytes=cap)
    for i in range(2):                                   # second pass: new payload through the same pipeline
        for key, a in payloads[i].items():
            if a.shape[0]:
                h_src[key].numpy()[:] = a.view(np.uint8)
        plan = hm.run()
        torch.cuda.synchronize()
        dm = None
        old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
        ov, _, _ = E.etc_cost_matrix(old, new)
        dm, _ = E.etc_sketch(ov)
        exp, T, _ = oracle_migrate(oo, on, dm.cpu().numpy(), payloads[i])
        assert np.array_equal(plan.traffic(), T)
        for key, e in exp.items():
            if e.shape[0]:
                got = h_dst[key].numpy().view(e.dtype)
                assert np.array_equal(got, e), (i, key)
    assert hm.h2d_bytes == sum(a.nbytes for a in payloads[0].values())


@pytest.mark.parametrize("name", ["s2", "s3", "s4"])
def test_chunked_migration_releases_and_matches(E, name):
    from paper_2607_04749_b200.host_pipeline import migrate_chunked
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    src_np = sharded_payload(oo, w["seed"], "stamp")
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    ov, need, hold = E.etc_cost_matrix(old, new)
    dm, _ = E.etc_sketch(ov)
    plan = E.etc_plan_create(old, new, dm, E.ETC_KIND_MAJOR)
    src = upload(src_np)
    dst, info = migrate_chunked(plan, new, src, 4 * 65536, fill=0x3C)
    torch.cuda.synchronize()
    assert not src                                       # every source buffer was released
    exp, _, _ = oracle_migrate(oo, on, dm.cpu().numpy(), src_np)
    for key, e in exp.items():
        if e.shape[0]:
            assert np.array_equal(download(dst[key], e.itemsize), e), key
    tot_old, tot_new = int(hold.sum().item()), int(need.sum().item())
    assert info["old_bytes"] == tot_old and info["new_bytes"] == tot_new
    assert info["staging_bytes"] <= 4 * 65536
    # one component at a time: the peak is below "everything old + everything new"
    assert info["peak_live_bytes"] < tot_old + tot_new + info["staging_bytes"]
    per_kind_old = {k: sum(a.nbytes for (d, kk), a in src_np.items() if kk == k) for k in on.kinds()}
    per_kind_new = {k: sum(e.nbytes for (n, kk), e in exp.items() if kk == k) for k in on.kinds()}
    live, peak = tot_old + info["staging_bytes"], 0
    for k in sorted(on.kinds()):
        live += per_kind_new[k]; peak = max(peak, live); live -= per_kind_old[k]
    assert info["peak_live_bytes"] == peak


@pytest.mark.parametrize("name", ["c1", "s2", "s3", "s4", "s5"])
def test_host_migration_uploads_only_what_the_plan_reads(E, name):
    """etc_upload_sources: the device copies of the old shards start poisoned and only the regions the plan's slices
    read are uploaded; the new shards still equal the oracle's, and the bytes that crossed PCIe are bounded below by
    the number of DISTINCT source elements the oracle's source rule reads (counted from O.source_of alone) and above by
    the whole old state."""
    from paper_2607_04749_b200.host_pipeline import HostMigration
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    payloads = [sharded_payload(oo, w["seed"] + i, "stamp" if i == 0 else "salted") for i in range(2)]
    h_src = _pinned(payloads[0])
    h_dst = {(n, k): torch.full((on.buffer_elems(n, k) * on.elem_bytes(k),), 0x77, dtype=torch.uint8).pin_memory()
             for n in range(on.n_dev) for k in on.kinds() if on.buffer_elems(n, k)}
    old = E.etc_layout_create(model, w["old"])
    d_src = E.alloc_buffers(old, fill=0xEE)
    hm = HostMigration(model, w["old"], w["new"], h_src, h_dst, max_staging_bytes=1 << 22, d_src=d_src, needed_only=True)
    for i in range(2):
        for key, a in payloads[i].items():
            if a.shape[0]:
                h_src[key].numpy()[:] = a.view(np.uint8)
        plan = hm.run()
        torch.cuda.synchronize()
        new = E.etc_layout_create(model, w["new"])
        ov, _, _ = E.etc_cost_matrix(old, new)
        dm = E.etc_sketch(ov)[0].cpu().numpy()
        exp, T, _ = oracle_migrate(oo, on, dm, payloads[i])
        assert np.array_equal(plan.traffic(), T)
        for key, e in exp.items():
            if e.shape[0]:
                assert np.array_equal(h_dst[key].numpy().view(e.dtype), e), (i, key)
    distinct = 0
    for k in on.kinds():
        seen = {o: np.zeros(oo.buffer_elems(o, k), bool) for o in range(oo.n_dev)}
        for n in range(on.n_dev):
            cnt = on.buffer_elems(n, k)
            if cnt:
                sd, sl = O.source_of(oo, on, dm, n, k, np.arange(cnt))
                for o in np.unique(sd):
                    seen[int(o)][sl[sd == o]] = True
        distinct += sum(int(v.sum()) for v in seen.values()) * on.elem_bytes(k)
    total_old = sum(a.nbytes for a in payloads[0].values())
    assert distinct <= hm.h2d_bytes <= total_old, (distinct, hm.h2d_bytes, total_old)
    print(f"{name}: uploaded {hm.h2d_bytes} of {total_old} old bytes; distinct source bytes {distinct}")
    if name in ("s2", "s3", "s5"):
        assert hm.h2d_bytes == distinct


@pytest.mark.parametrize("name", ["c1", "s2", "s3", "s4", "s4odd", "s5"])
@pytest.mark.parametrize("flags", [0, 1])
def test_host_migration_zero_copy(E, name, flags):
    """zero_copy=True: the pinned host shards are the source and destination tables of the copy kernels; there is no
    device copy of any shard.  New shards equal the oracle's; h2d / d2h byte counts are the payload."""
    from paper_2607_04749_b200.host_pipeline import HostMigration
    w = workload(name)
    model = w["model"]
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    payloads = [sharded_payload(oo, w["seed"] + i, "stamp" if i == 0 else "salted") for i in range(2)]
    h_src = _pinned(payloads[0])
    h_dst = {(n, k): torch.full((on.buffer_elems(n, k) * on.elem_bytes(k),), 0x77, dtype=torch.uint8).pin_memory()
             for n in range(on.n_dev) for k in on.kinds() if on.buffer_elems(n, k)}
    before = torch.cuda.memory_allocated()
    hm = HostMigration(model, w["old"], w["new"], h_src, h_dst, max_staging_bytes=4 * 65536, flags=flags, zero_copy=True)
    assert torch.cuda.memory_allocated() - before <= 4 * 65536 + 4096      # only the staging buffer lives on the device
    for i in range(2):
        for key, a in payloads[i].items():
            if a.shape[0]:
                h_src[key].numpy()[:] = a.view(np.uint8)
        plan = hm.run()
        torch.cuda.synchronize()
        old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
        dm = E.etc_sketch(E.etc_cost_matrix(old, new)[0])[0].cpu().numpy()
        exp, T, _ = oracle_migrate(oo, on, dm, payloads[i])
        assert np.array_equal(plan.traffic(), T)
        for key, e in exp.items():
            if e.shape[0]:
                assert np.array_equal(h_dst[key].numpy().view(e.dtype), e), (i, key)
    assert hm.h2d_bytes == int(T.sum()) == hm.d2h_bytes
