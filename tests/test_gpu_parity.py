"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, bit-exact.

Integer / byte work only, so every comparison is exact equality ("bit-exact fidelity").  Where several
results are correct (the sketch: several optimal device maps, reading A17) the objective value is compared and the map is
checked for validity; everything downstream is compared after feeding the GPU's own map to the oracle."""
from __future__ import annotations
import itertools
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload, tiny_models, tiny_parallel_cfgs, position_stamp
from oracle import oracle as O
from helpers import make_logical, shard_all, stamp_all, sharded_payload, oracle_migrate, oracle_overlap


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _oracle_layouts(w):
    return O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])


# ---------------------------------------------------------------------------------------------- (a1)+(a2) cost matrix
@pytest.mark.parametrize("name", ["c1", "s2", "s3", "s4", "s4odd", "s5", "s5b"])
def test_cost_matrix_vs_elementwise_oracle(E, name):
    w = workload(name)
    oo, on = _oracle_layouts(w)
    ov, need, hold = O.overlap(oo, on, method="elementwise" if name != "s5b" else "ranges")
    go, gn = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    for d in range(go.n_dev):
        for k in range(4):
            assert go.buffer_bytes(d, k) == oo.buffer_elems(d, k) * O.kind_bytes(w["model"], k)
    g_ov, g_need, g_hold = E.etc_cost_matrix(go, gn)
    assert np.array_equal(g_ov.cpu().numpy(), ov)
    assert np.array_equal(g_need.cpu().numpy(), need)
    assert np.array_equal(g_hold.cpu().numpy(), hold)


@pytest.mark.parametrize("name", ["c2", "c3", "c4", "c5", "c5b"])
def test_cost_matrix_full_size_configs(E, name):
    """BASELINE.json configs at full size (metadata only): GPU matrices == oracle's range routine (itself pinned to
    the element-wise definition on the small layouts and to SURVEY's independent byte counts)."""
    w = workload(name)
    oo, on = _oracle_layouts(w)
    ov, need, hold = O.overlap(oo, on, method="ranges")
    go, gn = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    g_ov, g_need, g_hold = E.etc_cost_matrix(go, gn)
    assert np.array_equal(g_ov.cpu().numpy(), ov)
    assert np.array_equal(g_need.cpu().numpy(), need)
    assert np.array_equal(g_hold.cpu().numpy(), hold)
    # sketch objective at full size, both solvers where applicable
    _, val = O.sketch_hungarian(ov)
    dm, lb = E.etc_sketch(g_ov, method=E.ETC_SKETCH_HUNGARIAN)
    dm = dm.cpu().numpy()
    assert int(lb.item()) == val
    assert len(set(dm.tolist())) == gn.n_dev and dm.min() >= 0 and dm.max() < ov.shape[1]
    assert sum(int(ov[n, dm[n]]) for n in range(gn.n_dev)) == val
    if ov.shape[1] <= 8:
        dm2, lb2 = E.etc_sketch(g_ov, method=E.ETC_SKETCH_EXHAUSTIVE)
        assert int(lb2.item()) == val


def test_cost_matrix_tiny_sweep(E):
    cfgs = tiny_parallel_cfgs(max_devices=8)
    rng = np.random.default_rng(11)
    ran = 0
    for name, model in tiny_models():
        for _ in range(40):
            a, b = cfgs[rng.integers(len(cfgs))], cfgs[rng.integers(len(cfgs))]
            try:
                oo, on = O.Layout(model, a), O.Layout(model, b)
            except O.OracleError as e:
                with pytest.raises(E.EtcError) as ge:            # same validation verdict on the GPU side
                    E.etc_layout_create(model, a); E.etc_layout_create(model, b)
                assert ge.value.code == e.code
                continue
            ov, need, hold = O.overlap(oo, on)
            go, gn = E.etc_layout_create(model, a), E.etc_layout_create(model, b)
            g = E.etc_cost_matrix(go, gn)
            assert np.array_equal(g[0].cpu().numpy(), ov), (name, a, b)
            assert np.array_equal(g[1].cpu().numpy(), need) and np.array_equal(g[2].cpu().numpy(), hold)
            ran += 1
    assert ran > 80


def test_cost_matrix_many_devices(E):
    """More than 8192 cells: etc_cost_matrix lists the (new stage, old stage) blocks that can overlap, clears the matrix and
    computes those blocks only.  Against the oracle's element-wise definition on layouts of 96-192 devices: even and
    uneven pipeline splits on either side, tied embeddings (the replica on the last stage overlaps stage 0), distributed
    optimizer, scale-out onto fresh devices and scale-in, PP1 on one side, both styles."""
    gpt = dict(style=0, n_layers=12, hidden=16, n_q_heads=4, n_kv_heads=4, head_dim=4, ffn_hidden=32, vocab=48,
               max_pos=6, tied=1, param_bytes=2, kinds=15)
    llama = dict(style=1, n_layers=12, hidden=16, n_q_heads=4, n_kv_heads=2, head_dim=4, ffn_hidden=24, vocab=32,
                 max_pos=0, tied=0, param_bytes=2, kinds=15)
    c = lambda tp, pp, dp, do=0, **kw: dict(dict(tp=tp, pp=pp, dp=dp, dist_opt=do), **kw)
    cases = [
        (gpt, c(2, 6, 8), c(2, 4, 12)),                          # 96 -> 96, stages cut differently
        (gpt, c(2, 12, 4), c(4, 3, 16, 1)),                      # 96 -> 192 (fresh devices), dist-opt
        (gpt, c(4, 4, 12, 1), c(2, 6, 8)),                       # 192 -> 96 scale-in
        (gpt, c(2, 4, 12, 0, pp_first=2, pp_last=4), c(1, 12, 8)),          # uneven old split
        (gpt, c(1, 1, 96), c(2, 6, 8, 0, pp_first=2)),           # PP1 on one side
        (llama, c(2, 6, 8), c(1, 12, 10)),                       # 96 -> 120, untied, GQA
        (llama, c(2, 3, 32, 1), c(2, 4, 16, 0, pp_last=3)),      # 192 -> 128
    ]
    for model, a, b in cases:
        oo, on = O.Layout(model, a), O.Layout(model, b)
        assert on.n_dev * max(oo.n_dev, on.n_dev) > 8192
        ov, need, hold = O.overlap(oo, on)
        go, gn = E.etc_layout_create(model, a), E.etc_layout_create(model, b)
        g = E.etc_cost_matrix(go, gn)
        assert np.array_equal(g[0].cpu().numpy(), ov), (a, b)
        assert np.array_equal(g[1].cpu().numpy(), need) and np.array_equal(g[2].cpu().numpy(), hold), (a, b)
        assert int(ov.sum()) > 0


def test_cost_matrix_mismatch_error(E):
    a = E.etc_layout_create(dict(tiny_models())["gpt_t"], dict(tp=1, pp=1, dp=1, dist_opt=0))
    b = E.etc_layout_create(dict(tiny_models())["gpt_u"], dict(tp=1, pp=1, dp=1, dist_opt=0))
    out = torch.zeros(4, dtype=torch.int64, device="cuda")
    with pytest.raises(E.EtcError) as e:
        E.etc_cost_matrix(a, b, out=(out, out, out))
    assert e.value.code == -3


# ---------------------------------------------------------------------------------------------- (a3) sketch
def _check_sketch(E, ov, avail=None, methods=None):
    n, P = ov.shape
    g = torch.from_numpy(np.ascontiguousarray(ov, np.int64)).cuda()
    av = None if avail is None else torch.from_numpy(avail.astype(np.uint8)).cuda()
    if P <= 8:
        _, ref, _ = O.sketch_bruteforce(ov, avail)
    else:
        ref = O.sketch_hungarian(ov, avail)[1]
    methods = methods or ([E.ETC_SKETCH_EXHAUSTIVE, E.ETC_SKETCH_HUNGARIAN] if P <= 8 else [E.ETC_SKETCH_HUNGARIAN])
    for m in methods:
        dm, lb = E.etc_sketch(g, avail=av, method=m)
        dm = dm.cpu().numpy(); lb = int(lb.item())
        assert lb == ref, (m, lb, ref)
        assert len(set(dm.tolist())) == n and dm.min() >= 0 and dm.max() < P
        if avail is not None:
            assert all(avail[p] for p in dm)
        assert sum(int(ov[i, dm[i]]) for i in range(n)) == lb


def test_sketch_random_matrices(E):
    rng = np.random.default_rng(3)
    for trial in range(80):
        P = int(rng.integers(1, 9)); n = int(rng.integers(1, P + 1))
        if trial % 3 == 0:
            ov = rng.integers(0, 1000, size=(n, P))
        elif trial % 3 == 1:
            ov = rng.integers(0, 3, size=(n, P)) * 10**11               # heavy ties, large values
        else:
            ov = np.zeros((n, P), np.int64); ov[:, : max(1, P // 2)] = rng.integers(0, 50, size=(n, max(1, P // 2)))
        _check_sketch(E, ov.astype(np.int64))
        avail = (rng.random(P) < 0.8)
        if avail.sum() >= n:
            _check_sketch(E, ov.astype(np.int64), avail)


def test_sketch_large_random_and_structured(E):
    from scipy.optimize import linear_sum_assignment
    rng = np.random.default_rng(4)
    for n, P in [(12, 16), (32, 32), (100, 130), (384, 512), (1000, 1024), (2048, 2048), (7, 2000)]:
        ov = rng.integers(0, 10**9, size=(n, P)).astype(np.int64)
        if n == 32:
            ov = (ov // 10**8) * 10**8                                   # ties
        g = torch.from_numpy(ov).cuda()
        dm, lb = E.etc_sketch(g, method=E.ETC_SKETCH_HUNGARIAN)
        r, c = linear_sum_assignment(ov, maximize=True)                  # the routine the paper calls
        assert int(lb.item()) == int(ov[r, c].sum()), (n, P)
        dm = dm.cpu().numpy()
        assert len(set(dm.tolist())) == n
        assert sum(int(ov[i, dm[i]]) for i in range(n)) == int(lb.item())


def test_sketch_row_maximum_certificate(E):
    """P > 32: sketch_tight_kernel tries to give every row one of its maximal columns (then the row-maximum bound proves
    optimality) and otherwise hands over to the Hungarian kernel.  Either way the objective must equal the oracle's /
    SciPy's: matrices where the certificate holds (replicated maxima as in DP groups, zero rows taking leftover columns,
    masked columns), where greedy needs the most-constrained-first order, where it cannot hold (contended maxima), and
    an infeasible mask."""
    from scipy.optimize import linear_sum_assignment
    rng = np.random.default_rng(11)

    def check(ov, avail=None):
        g = torch.from_numpy(np.ascontiguousarray(ov, np.int64)).cuda()
        av = None if avail is None else torch.from_numpy(avail.astype(np.uint8)).cuda()
        dm, lb = E.etc_sketch(g, avail=av, method=E.ETC_SKETCH_HUNGARIAN)
        dm = dm.cpu().numpy(); lb = int(lb.item())
        m = ov.copy()
        if avail is not None:
            m = m[:, avail]
        if m.shape[1] < m.shape[0]:
            assert lb == -1 and (dm == -1).all()
            return
        r, c = linear_sum_assignment(m, maximize=True)
        assert lb == int(m[r, c].sum()), (ov.shape, lb, int(m[r, c].sum()))
        assert len(set(dm.tolist())) == ov.shape[0] and dm.min() >= 0 and dm.max() < ov.shape[1]
        if avail is not None:
            assert all(avail[p] for p in dm)
        assert sum(int(ov[i, dm[i]]) for i in range(ov.shape[0])) == lb

    for n, P, rep in [(48, 64, 4), (96, 128, 4), (384, 512, 4), (200, 1000, 5), (1024, 1024, 1), (33, 40, 8)]:
        # groups of `rep` equal columns (old DP replicas); every row's maximum sits on one group, <= rep rows per group
        groups = P // rep
        ov = np.zeros((n, P), np.int64)
        for i in range(n):
            gi = (i // rep) % groups if rep > 1 else i % groups
            ov[i, gi * rep:(gi + 1) * rep] = 10**9 + 7 * gi
            ov[i, rng.integers(0, P, size=3)] += rng.integers(0, 1000, size=3)     # noise below / inside the maxima
        check(ov)
        # fresh ranks: the last quarter of the rows overlaps nothing (scale-out)
        ov2 = ov.copy(); ov2[n - n // 4:] = 0
        check(ov2)
        # masked columns (pre-emption): the certificate may or may not survive
        avail = rng.random(P) < 0.9
        check(ov, avail)
    # most-constrained-first: row 0 ties on columns {0,1}, row 1 wants column 0 only
    ov = np.zeros((40, 64), np.int64)
    ov[0, 0] = ov[0, 1] = 5; ov[1, 0] = 5
    for i in range(2, 40):
        ov[i, i + 3] = 9
    check(ov)
    # contended maxima: all rows want column 0 -> no certificate, the Hungarian kernel decides
    ov = rng.integers(0, 100, size=(50, 70)).astype(np.int64); ov[:, 0] = 10**6
    check(ov)
    # dense random (fallback) and heavy ties
    check(rng.integers(0, 10**9, size=(60, 90)).astype(np.int64))
    check((rng.integers(0, 3, size=(64, 64)) * 10**11).astype(np.int64))
    # infeasible: fewer usable columns than rows
    avail = np.zeros(64, bool); avail[:10] = True
    check(rng.integers(0, 9, size=(40, 64)).astype(np.int64), avail)


def test_sketch_infeasible_and_errors(E):
    ov = torch.ones((3, 4), dtype=torch.int64, device="cuda")
    av = torch.tensor([1, 0, 0, 1], dtype=torch.uint8, device="cuda")
    for m in (E.ETC_SKETCH_EXHAUSTIVE, E.ETC_SKETCH_HUNGARIAN):
        dm, lb = E.etc_sketch(ov, avail=av, method=m)
        assert int(lb.item()) == -1 and (dm.cpu().numpy() == -1).all()
    big = torch.zeros((2, 9), dtype=torch.int64, device="cuda")
    with pytest.raises(E.EtcError) as e:
        E.etc_sketch(big, method=E.ETC_SKETCH_EXHAUSTIVE)
    assert e.value.code == -5


# ---------------------------------------------------------------------------------------------- (a4)-(a6) plan + migrate
def _check_migration(E, model, old_cfg, new_cfg, seed, device_map=None, flags=0, payload="stamp"):
    from gpu_helpers import run_gpu_migration
    oo, on = O.Layout(model, old_cfg), O.Layout(model, new_cfg)
    src = sharded_payload(oo, seed, payload)
    g = run_gpu_migration(model, old_cfg, new_cfg, src, device_map=device_map, flags=flags)
    ov, need, hold = oracle_overlap(oo, on)
    assert np.array_equal(g["overlap"], ov) and np.array_equal(g["need"], need) and np.array_equal(g["hold"], hold)
    dm = g["device_map"]
    if device_map is None:
        P = ov.shape[1]
        ref = O.sketch_bruteforce(ov)[1] if P <= 8 else O.sketch_hungarian(ov)[1]
        assert g["local_bytes"] == ref
    # oracle migration with the GPU's own map (A17)
    dst, T, _ = oracle_migrate(oo, on, dm, src)
    st = g["plan"].stats
    assert np.array_equal(g["plan"].traffic(), T)
    local = int(np.trace(T)); remote = int(T.sum() - np.trace(T))
    assert st.local_bytes == local and st.remote_bytes == remote and local + remote == int(need.sum())
    assert st.staged_bytes == (local + remote if flags & E.ETC_ALL_STAGED else (0 if flags & E.ETC_ALL_DIRECT else remote))
    assert not (flags & E.ETC_ALL_DIRECT) or st.staging_bytes == 0
    for key, exp in dst.items():
        got = g["dst"][key]
        assert got.shape == exp.shape, key
        assert np.array_equal(got, exp), (key, int((got != exp).sum()))
    # slice table: every destination byte written exactly once, staging segments disjoint and inside the buffer
    cover = {key: np.zeros(v.shape[0] * v.itemsize, np.uint8) for key, v in dst.items()}
    stg = np.zeros(max(st.staging_bytes, 1), np.uint8)
    from numpy.lib.stride_tricks import as_strided
    for which in (0, 1):
        for s in g["plan"].slices(which):
            key = (int(s["dst_rank"]), int(s["kind"]))
            nrows, rb, a0 = int(s["nrows"]), int(s["row_bytes"]), int(s["dst_off"])
            pitch = int(s["dst_stride"]) if nrows > 1 else rb
            assert pitch >= rb and a0 >= 0 and a0 + (nrows - 1) * pitch + rb <= cover[key].shape[0], key
            as_strided(cover[key][a0:], shape=(nrows, rb), strides=(pitch, 1))[...] += 1     # rows x row_bytes at the pitch
            if which == 0:
                b0 = int(s["stg_off"])
                assert b0 >= 0 and b0 + nrows * rb <= stg.shape[0]
                stg[b0:b0 + nrows * rb] += 1                                                  # packed back to back
            assert int(s["dst_phys"]) == int(dm[int(s["dst_rank"])])
    for key, c in cover.items():
        assert (c == 1).all(), key
    assert stg.max() <= 1 and int(stg.sum()) == st.staged_bytes
    return g


@pytest.mark.parametrize("flags", [0, 1])
def test_migrate_config1(E, flags):
    w = workload("c1")
    _check_migration(E, w["model"], w["old"], w["new"], w["seed"], flags=flags, payload="values")
    _check_migration(E, w["model"], w["old"], w["new"], w["seed"], flags=flags, payload="stamp")


@pytest.mark.parametrize("name", ["s2", "s2odd", "s3", "s4", "s4odd", "s5", "sx64", "sxodd"])
@pytest.mark.parametrize("flags", [0, 1, 2, 3, 4, 6])        # 2, 3: + ETC_KIND_MAJOR; 4, 6: ETC_ALL_DIRECT (nothing staged)
def test_migrate_scaled_configs(E, name, flags):
    w = workload(name)
    _check_migration(E, w["model"], w["old"], w["new"], w["seed"], flags=flags)


@pytest.mark.parametrize("hidden", [66, 130, 258])
def test_migrate_misaligned_wide_rows(E, hidden):
    """Rows of 264 ... 1032 bytes whose addresses are only 4- or 8-byte aligned and whose pitches are not multiples of 16
    (the source / destination phase modulo 16 changes from row to row), with distributed-optimizer cuts on both sides:
    the re-aligning staged copy path (16-byte loads and stores through a phase-shifted tile) against the oracle."""
    m = dict(workload("s2")["model"], hidden=hidden, n_q_heads=4, n_kv_heads=4, head_dim=16, ffn_hidden=4 * hidden,
             vocab=516, max_pos=33, n_layers=4)
    old_c, new_c = dict(tp=2, pp=2, dp=2, dist_opt=1), dict(tp=4, pp=1, dp=2, dist_opt=1)
    rng = np.random.default_rng(hidden)
    for flags in (0, 1):
        _check_migration(E, m, old_c, new_c, 300 + hidden, flags=flags)
    _check_migration(E, m, old_c, new_c, 301 + hidden, device_map=rng.permutation(8).astype(np.int32), flags=3, payload="values")
    _check_migration(E, m, new_c, old_c, 302 + hidden, flags=1)


def test_migrate_identity_map_and_arbitrary_maps(E):
    rng = np.random.default_rng(8)
    w = workload("s3")                       # 16 -> 12: identity on the first 12, then random injective maps
    _check_migration(E, w["model"], w["old"], w["new"], 5, device_map=np.arange(12, dtype=np.int32))
    for _ in range(2):
        _check_migration(E, w["model"], w["old"], w["new"], 5, device_map=rng.permutation(16)[:12].astype(np.int32))
    w = workload("s4")                       # 16 -> 32 (fresh devices), dist-opt, tied replica on another stage
    for _ in range(2):
        _check_migration(E, w["model"], w["old"], w["new"], 6, device_map=rng.permutation(32).astype(np.int32))


def test_migrate_tiny_sweep(E):
    cfgs = tiny_parallel_cfgs(max_devices=8)
    rng = np.random.default_rng(12)
    ran = 0
    models = dict(tiny_models())
    for name, model in models.items():
        for t in range(30):
            a, b = cfgs[rng.integers(len(cfgs))], cfgs[rng.integers(len(cfgs))]
            try:
                O.Layout(model, a); O.Layout(model, b)
            except O.OracleError:
                continue
            dm = None
            if t % 3 == 2:                   # arbitrary (non-optimal) injective map
                nn, no = b["tp"] * b["pp"] * b["dp"], a["tp"] * a["pp"] * a["dp"]
                dm = rng.permutation(max(nn, no))[:nn].astype(np.int32)
            _check_migration(E, model, a, b, 1000 + t, device_map=dm, flags=t % 2)
            ran += 1
    assert ran > 60


def test_position_stamped_payload_names_sources(E):
    """P9: values say which old buffer and position they came from; compare with the oracle's source rule."""
    from gpu_helpers import run_gpu_migration
    w = workload("s4")
    oo, on = _oracle_layouts(w)
    src = stamp_all(oo)
    g = run_gpu_migration(w["model"], w["old"], w["new"], src)
    dm = g["device_map"]
    for n in range(on.n_dev):
        for k in on.kinds():
            cnt = on.buffer_elems(n, k)
            if not cnt:
                continue
            sd, sl = O.source_of(oo, on, dm, n, k, np.arange(cnt))
            es = on.elem_bytes(k)
            exp = np.zeros(cnt, g["dst"][(n, k)].dtype)
            for o in np.unique(sd):
                sel = sd == o
                exp[sel] = position_stamp(int(o), k, oo.buffer_elems(int(o), k), es)[sl[sel]]
            assert np.array_equal(g["dst"][(n, k)], exp), (n, k)


def test_plan_errors(E):
    w = workload("c1")
    old, new = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    for bad in ([0, 0, 1, 2], [0, 1, 2, 4], [-1, 1, 2, 3]):
        with pytest.raises(E.EtcError) as e:
            E.etc_plan_create(old, new, np.array(bad, np.int32))
        assert e.value.code == -4
        with pytest.raises(E.EtcError) as e:
            E.etc_plan_create(old, new, torch.tensor(bad, dtype=torch.int32, device="cuda"))
        assert e.value.code == -4
    plan = E.etc_plan_create(old, new, np.arange(4, dtype=np.int32))
    dst = E.alloc_buffers(new)
    src = E.alloc_buffers(old)
    with pytest.raises(E.EtcError):                      # staging missing although bytes must be staged
        E.etc_migrate(plan, src, dst, None)
    del src[(0, 0)]
    stg = torch.empty(plan.stats.staging_bytes, dtype=torch.uint8, device="cuda")
    with pytest.raises(E.EtcError):                      # a needed source buffer is NULL
        E.etc_migrate(plan, src, dst, stg)


def test_empty_and_degenerate_layouts(E):
    """Single device -> single device (everything local, nothing staged) and a 1 -> many broadcast."""
    model = dict(tiny_models())["gpt_t"]
    one = dict(tp=1, pp=1, dp=1, dist_opt=0)
    g = _check_migration(E, model, one, one, 3)
    assert g["plan"].stats.staging_bytes == 0 and g["plan"].stats.n_slices_staged == 0
    _check_migration(E, model, one, dict(tp=2, pp=2, dp=2, dist_opt=1), 3)
    _check_migration(E, model, dict(tp=2, pp=2, dp=2, dist_opt=1), one, 3)
