"""-m gpu: BASELINE.json configs at FULL size, in the launch configuration bench.py times (whole path, LOCAL_DIRECT with
the GPU's own optimal sketch; plus ALL_STAGED for the bench workload).  The element-wise oracle cannot enumerate 20-56 GB
in a test, so outputs are SAMPLED: every sampled destination element is computed one by one by the oracle (source rule A6
-> position-stamped source value), with samples placed at random positions, at buffer ends and at the first / last
element of slices (where an off-by-one would show).  Properties that hold at any size are checked in full: traffic matrix
== oracle's row-level traffic, byte totals, and "every destination byte is written" (two runs with different poison)."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload, position_stamp_at, position_stamp_torch
from oracle import oracle as O


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _stamped_sources(lay, model, dev):
    src = {}
    for d in range(lay.n_dev):
        for k in lay.kinds():
            nb = lay.buffer_bytes(d, k)
            if nb:
                es = 4 if k else model["param_bytes"]
                src[(d, k)] = position_stamp_torch(d, k, nb // es, es, dev).view(torch.uint8)
    return src


def _run(E, name, flags, poison_runs):
    w = workload(name)
    model = w["model"]
    dev = torch.device("cuda", torch.cuda.current_device())
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    ov, need, hold = E.etc_cost_matrix(old, new)
    dm, lb = E.etc_sketch(ov)
    o_ov, o_need, o_hold = O.overlap(oo, on, method="ranges")
    assert np.array_equal(ov.cpu().numpy(), o_ov) and np.array_equal(need.cpu().numpy(), o_need)
    assert int(lb.item()) == O.sketch_hungarian(o_ov)[1]
    plan = E.etc_plan_create(old, new, dm, flags)
    assert plan.validate() == 0
    st = plan.stats
    dmap = dm.cpu().numpy()
    T = plan.traffic()
    # properties at any size
    assert st.local_bytes + st.remote_bytes == int(o_need.sum())
    assert st.local_bytes == int(lb.item()) == int(np.trace(T))
    for n in range(on.n_dev):
        assert int(T[:, dmap[n]].sum()) == int(o_need[n])
    assert (T.sum(axis=1)[: oo.n_dev] <= o_hold[: oo.n_dev] * max(1, on.n_dev)).all()
    src = _stamped_sources(old, model, dev)
    dst = E.alloc_buffers(new, dev)
    staging = torch.empty(max(st.staging_bytes, 16), dtype=torch.uint8, device=dev)
    prev = None
    for poison in poison_runs:
        for t in dst.values():
            t.fill_(poison)
        staging.fill_(poison)
        E.etc_migrate(plan, src, dst, staging)
        torch.cuda.synchronize()
        if prev is not None:                       # every byte written: identical results under different poison
            for key, t in dst.items():
                assert torch.equal(t, prev[key]), key
        if len(poison_runs) > 1 and prev is None:
            prev = {k: t.clone() for k, t in dst.items()}
    del prev
    # sampled element-by-element parity
    rng = np.random.default_rng(20260704)
    sl_all = [plan.slices(0), plan.slices(1)]
    checked = 0
    for n in range(on.n_dev):
        for k in on.kinds():
            cnt = on.buffer_elems(n, k)
            if not cnt:
                continue
            es = on.elem_bytes(k)
            idx = [rng.integers(0, cnt, size=600), np.arange(min(cnt, 48)), np.arange(max(0, cnt - 48), cnt)]
            for sl in sl_all:                      # first / last element of (up to 150) slices landing in this buffer
                m = sl[(sl["dst_rank"] == n) & (sl["kind"] == k)]
                if len(m) > 150:
                    m = m[rng.choice(len(m), 150, replace=False)]
                first = m["dst_off"] // es
                last = (m["dst_off"] + (m["nrows"].astype(np.int64) - 1) * m["dst_stride"] + m["row_bytes"]) // es - 1
                idx += [first, last, np.clip(first - 1, 0, cnt - 1), np.clip(last + 1, 0, cnt - 1)]
            idx = np.unique(np.concatenate(idx).astype(np.int64))
            sd, sl_ = O.source_of(oo, on, dmap, n, k, idx)
            exp = np.zeros(idx.shape[0], np.uint16 if es == 2 else np.uint32)
            for o in np.unique(sd):
                sel = sd == o
                exp[sel] = position_stamp_at(int(o), k, sl_[sel], es)
            view = dst[(n, k)].view(torch.int16 if es == 2 else torch.int32)
            got = view[torch.from_numpy(idx).to(dev)].cpu().numpy().view(exp.dtype)
            assert np.array_equal(got, exp), (name, n, k, int((got != exp).sum()))
            checked += idx.shape[0]
    return checked


def test_fullsize_c2_local_direct_and_all_staged(E):
    assert _run(E, "c2", E.ETC_LOCAL_DIRECT, [0x00, 0xFF]) > 20000
    assert _run(E, "c2", E.ETC_ALL_STAGED, [0x5A]) > 20000


def test_fullsize_c3(E):
    assert _run(E, "c3", E.ETC_LOCAL_DIRECT, [0x00, 0xFF]) > 30000


def test_fullsize_c4(E):
    torch.cuda.empty_cache()
    assert _run(E, "c4", E.ETC_LOCAL_DIRECT, [0xA5]) > 50000


def test_fullsize_c5(E):
    torch.cuda.empty_cache()
    assert _run(E, "c5", E.ETC_LOCAL_DIRECT, [0xA5]) > 20000
