"""etc_sketch_static: the migration sketch for callers that cannot allocate device memory.

Why it exists (include/etc.h has the full text): the sketch is computed while a training job is being reconfigured, i.e.
when HBM is at its fullest and the trainer's own caching allocator holds whatever is left; a recovery handler must not
wait on the allocator either, and some processes run under a fixed device-memory budget.  For those callers
etc_sketch_static keeps its work area (28 KB, P <= 1024) in an array that is part of libetc.so's device image instead of
taking it from CUDA's stream-ordered pool as etc_sketch does.

What is checked here: on the same matrices, etc_sketch_static returns exactly what the existing path
etc_sketch(method=ETC_SKETCH_HUNGARIAN) returns — the sketch is integer work and both paths are deterministic, so the
tolerance is the one every sketch test in this repository uses: equality, of the objective AND of the device map — on two
calls in a row through the shared work area (the second with a smaller matrix, so that rows left behind by the first call
lie behind its own), then again with the first matrix; that the stream-ordered pool does not grow across the calls; and
that a P beyond the limit is refused with a readable message before anything is launched.

This file is named to be collected last: it must pass on its own in a fresh process (where its first call does the one-time
address look-up) and after every other GPU test has used the library."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _replicated_maxima(rng, n, P, rep):
    """Overlap matrix of a reconfiguration with `rep` old DP replicas: groups of `rep` equal columns, every row's maximum on
    one group (the row-maximum certificate holds), a little noise elsewhere."""
    groups = P // rep
    ov = np.zeros((n, P), np.int64)
    for i in range(n):
        gi = (i // rep) % groups
        ov[i, gi * rep:(gi + 1) * rep] = 10**9 + 7 * gi
        ov[i, rng.integers(0, P, size=3)] += rng.integers(0, 1000, size=3)
    return ov


def _cases():
    rng = np.random.default_rng(2607)
    first = _replicated_maxima(rng, 384, 512, 4)                       # certificate holds; the 512 -> 384-device shape
    avail = rng.random(512) < 0.9                                      # pre-empted devices
    second = rng.integers(0, 10**9, size=(60, 90)).astype(np.int64)    # dense random: certificate fails, CTA search decides
    contended = rng.integers(0, 100, size=(50, 70)).astype(np.int64); contended[:, 0] = 10**6
    full = _replicated_maxima(rng, 1024, 1024, 1)                      # the largest size the work area holds
    small = rng.integers(0, 1000, size=(12, 16)).astype(np.int64)      # P <= 32: warp search, no work area at all
    few = np.zeros(64, bool); few[:10] = True                          # infeasible: 40 rows, 10 usable columns
    return [(first, None), (second, None), (first, avail), (contended, None), (full, None), (small, None),
            (rng.integers(0, 9, size=(40, 64)).astype(np.int64), few), (first, None)]


def test_static_sketch_equals_existing_path_on_consecutive_calls(E):
    dev = torch.device("cuda", torch.cuda.current_device())
    cases = [(torch.from_numpy(ov).to(dev), None if av is None else torch.from_numpy(av.astype(np.uint8)).to(dev))
             for ov, av in _cases()]
    # reference results from the existing (allocating) path
    ref = [tuple(t.clone() for t in E.etc_sketch(ov, avail=av, method=E.ETC_SKETCH_HUNGARIAN)) for ov, av in cases]
    # the caller owns the outputs: allocate them before the calls under test, poisoned
    outs = [(torch.full((ov.shape[0],), -7, dtype=torch.int32, device=dev), torch.full((1,), -7, dtype=torch.int64, device=dev))
            for ov, _ in cases]
    torch.cuda.synchronize()
    E.etc_sketch_static(cases[0][0], outs[0], avail=cases[0][1])       # first call on this device: one-time address look-up
    torch.cuda.synchronize()
    pool_before = _pool_reserved()
    launches_before = E.kernel_launches()
    for (ov, av), out in zip(cases[1:], outs[1:]):                     # back to back on one stream, no sync in between
        E.etc_sketch_static(ov, out, avail=av)
    torch.cuda.synchronize()
    assert E.kernel_launches() > launches_before                       # the library's kernels ran (no other path exists)
    assert _pool_reserved() == pool_before                             # nothing was taken from the stream-ordered pool
    for i, ((ov, av), (dm, lb), (rdm, rlb)) in enumerate(zip(cases, outs, ref)):
        assert int(lb.item()) == int(rlb.item()), (i, tuple(ov.shape))
        assert torch.equal(dm, rdm), (i, tuple(ov.shape))
        n, P = ov.shape
        if int(rlb.item()) >= 0:                                       # and the map is a sketch in its own right
            m = dm.cpu().numpy()
            assert len(set(m.tolist())) == n and m.min() >= 0 and m.max() < P
            assert int(ov.cpu().numpy()[np.arange(n), m].sum()) == int(lb.item())
    assert int(ref[6][1].item()) == -1 and bool((outs[6][0] == -1).all())   # the infeasible case says so on both paths


def _pool_reserved():
    """Bytes the device's default stream-ordered pool (the one etc_sketch draws from) has reserved from the driver."""
    from cuda.bindings import runtime as rt
    err, pool = rt.cudaDeviceGetDefaultMemPool(torch.cuda.current_device())
    assert int(err) == 0
    err, v = rt.cudaMemPoolGetAttribute(pool, rt.cudaMemPoolAttr.cudaMemPoolAttrReservedMemCurrent)
    assert int(err) == 0
    return int(v)


def test_static_sketch_refuses_sizes_beyond_its_work_area(E):
    assert E.ETC_SKETCH_STATIC_MAX_P == 1024 and E.ETC_SKETCH_STATIC_SCRATCH_BYTES == 1024 * (8 + 4 + 16)
    P = E.ETC_SKETCH_STATIC_MAX_P + 1
    ov = torch.zeros((2, P), dtype=torch.int64, device="cuda")
    out = (torch.full((2,), -7, dtype=torch.int32, device="cuda"), torch.full((1,), -7, dtype=torch.int64, device="cuda"))
    before = E.kernel_launches()
    with pytest.raises(E.EtcError) as e:
        E.etc_sketch_static(ov, out)
    assert e.value.code == -5 and "ETC_SKETCH_STATIC_MAX_P" in str(e.value) and "1025" in str(e.value)
    torch.cuda.synchronize()
    assert E.kernel_launches() == before and int(out[1].item()) == -7 and bool((out[0] == -7).all())   # nothing ran
