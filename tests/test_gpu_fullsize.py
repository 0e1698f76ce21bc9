"""-m gpu: BASELINE.json configs c2-c5 at FULL size, in the launch configuration bench.py times (whole path, the GPU's own
optimal sketch, LOCAL_DIRECT, address-ordered launches; every slice staged, ALL_STAGED; and LOCAL_DIRECT with the launches
in list order, ETC_NO_REORDER).  EXHAUSTIVE: the oracle's element-wise migration
(oracle/etc_oracle.c orc_migrate_range: global_of -> holders_of -> source rule A6 -> one element copied) is run over EVERY
element of EVERY new shard buffer on all host cores, from a host copy of the position-stamped old state, and every new
shard buffer the CUDA path produced is compared with it byte for byte ("bit-exact fidelity"; north_star:
bit-exact new-layout shards on all five configs; c1 is exhaustive in test_gpu_parity.py).  The destination buffers and the
staging buffer start poisoned, so equality also proves that every byte was written.  Properties that hold at any size are
checked as well: cost matrix == the oracle's row-level routine, sketch objective == the oracle's Hungarian, traffic matrix
identities, byte totals, device-side bounds check of every copy work item."""
from __future__ import annotations
import os
from concurrent.futures import ThreadPoolExecutor
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload, position_stamp, position_stamp_torch
from oracle import oracle as O

CHUNK = 1 << 22            # elements per oracle task


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


def _oracle_expected(oo, on, dmap, h_src, pool):
    """{(n, kind): numpy array} — every element of every new buffer through the oracle's element-wise migration."""
    exp, tasks = {}, []
    for n in range(on.n_dev):
        for k in on.kinds():
            cnt = on.buffer_elems(n, k)
            if not cnt:
                continue
            a = np.empty(cnt, np.uint16 if on.elem_bytes(k) == 2 else np.uint32)
            exp[(n, k)] = a
            tasks += [(n, k, l0, min(cnt, l0 + CHUNK)) for l0 in range(0, cnt, CHUNK)]

    def one(t):
        n, k, l0, l1 = t
        O.migrate_range(oo, on, dmap, n, k, l0, l1, h_src, exp[(n, k)])      # writes elements [l0, l1) of the buffer

    list(pool.map(one, tasks))
    return exp


def _exhaustive(E, name, modes):
    w = workload(name)
    model = w["model"]
    dev = torch.device("cuda", torch.cuda.current_device())
    torch.cuda.empty_cache()
    oo, on = O.Layout(model, w["old"]), O.Layout(model, w["new"])
    old, new = E.etc_layout_create(model, w["old"]), E.etc_layout_create(model, w["new"])
    ov, need, hold = E.etc_cost_matrix(old, new)
    dm, lb = E.etc_sketch(ov)
    o_ov, o_need, o_hold = O.overlap(oo, on, method="ranges")
    assert np.array_equal(ov.cpu().numpy(), o_ov) and np.array_equal(need.cpu().numpy(), o_need)
    assert int(lb.item()) == O.sketch_hungarian(o_ov)[1]
    dmap = dm.cpu().numpy()

    src = _stamped_sources(old, model, dev)
    # host copy of the old state for the oracle (the generator's output, not the CUDA path's); spot-checked against the
    # numpy generator so that both sides start from the same bytes
    h_src = {key: t.cpu().numpy().view(np.uint16 if (key[1] == 0 and model["param_bytes"] == 2) else np.uint32)
             for key, t in src.items()}
    for key in list(h_src)[:: max(1, len(h_src) // 6)]:
        a = h_src[key]
        assert np.array_equal(a[-4096:], position_stamp(key[0], key[1], a.shape[0], a.itemsize)[-4096:])
    with ThreadPoolExecutor(os.cpu_count() or 1) as pool:
        exp = _oracle_expected(oo, on, dmap, h_src, pool)
    del h_src

    dst = E.alloc_buffers(new, dev)
    checked = 0
    for flags, poison in modes:
        plan = E.etc_plan_create(old, new, dm, flags)
        assert plan.validate() == 0
        st = plan.stats
        T = plan.traffic()
        assert st.local_bytes + st.remote_bytes == int(o_need.sum())
        assert st.local_bytes == int(lb.item()) == int(np.trace(T))
        for n in range(on.n_dev):
            assert int(T[:, dmap[n]].sum()) == int(o_need[n])
        assert (T.sum(axis=1)[: oo.n_dev] <= o_hold[: oo.n_dev] * max(1, on.n_dev)).all()
        try:
            staging = torch.full((max(st.staging_bytes, 16),), poison, dtype=torch.uint8, device=dev)
        except torch.cuda.OutOfMemoryError:
            pytest.skip(f"{name}: staging of {st.staging_bytes} bytes does not fit beside the shards")
        for t in dst.values():
            t.fill_(poison)
        E.etc_migrate(plan, src, dst, staging)
        torch.cuda.synchronize()
        del staging
        for key, a in exp.items():                        # EVERY byte of EVERY new buffer
            want = torch.from_numpy(a.view(np.uint8)).to(dev)
            assert torch.equal(dst[key], want), (name, flags, key)
            checked += a.shape[0]
            del want
        del plan
        torch.cuda.empty_cache()
    total = sum(on.buffer_elems(n, k) for n in range(on.n_dev) for k in on.kinds())
    assert checked == total * len(modes)
    return checked


def test_fullsize_c2_exhaustive(E):
    _exhaustive(E, "c2", [(E.ETC_LOCAL_DIRECT, 0x00), (E.ETC_ALL_STAGED, 0xFF), (E.ETC_LOCAL_DIRECT | E.ETC_NO_REORDER, 0x3C)])


def test_fullsize_c3_exhaustive(E):
    _exhaustive(E, "c3", [(E.ETC_LOCAL_DIRECT, 0x00), (E.ETC_ALL_STAGED, 0xFF), (E.ETC_LOCAL_DIRECT | E.ETC_NO_REORDER, 0x3C)])


def test_fullsize_c4_exhaustive(E):
    _exhaustive(E, "c4", [(E.ETC_LOCAL_DIRECT, 0xA5), (E.ETC_ALL_STAGED, 0x5A), (E.ETC_LOCAL_DIRECT | E.ETC_NO_REORDER, 0x3C)])


def test_fullsize_c5_exhaustive(E):
    _exhaustive(E, "c5", [(E.ETC_LOCAL_DIRECT, 0xA5), (E.ETC_ALL_STAGED, 0x5A), (E.ETC_LOCAL_DIRECT | E.ETC_NO_REORDER, 0x3C)])


@pytest.mark.parametrize("name", ["x64", "x64r", "x128", "xodd"])
def test_fullsize_stress_workloads_exhaustive(E, name):
    """The copy-kernel stress workloads at FULL size: rows of 64-512 B on the source side (x64, x128) or
    the destination side (x64r), and 2-byte-aligned long rows (xodd: the byte-phase re-aligning path).  DESIGN.md quotes their
    copy rates, so every byte they write is compared with the oracle too — direct + staged, and every slice staged."""
    _exhaustive(E, name, [(E.ETC_LOCAL_DIRECT, 0xA5), (E.ETC_ALL_STAGED, 0x5A)])
