"""-m gpu parity of failure-aware sourcing (f4, reading A26): masked cost matrix, sketch that avoids or
reuses failed slots, plan + migrate with a failure mask — bit-exact against the oracle; unrecoverable cases."""
from __future__ import annotations
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload, tiny_models, tiny_parallel_cfgs
from oracle import oracle as O
from helpers import make_logical, shard_all, stamp_all
from gpu_helpers import upload, download


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


def _survivable_mask(cfg, rng):
    tp, pp, dp = cfg["tp"], cfg["pp"], cfg["dp"]
    f = np.zeros(tp * pp * dp, np.uint8)
    for s in range(pp):
        for r in range(tp):
            for d in rng.permutation(dp)[: int(rng.integers(0, dp))]:
                f[r + tp * (int(d) + dp * s)] = 1
    return f


def _run(E, model, old_c, new_c, f, seed, flags=0, device_map=None, avoid_failed=True, payload="stamp"):
    oo, on = O.Layout(model, old_c), O.Layout(model, new_c)
    src_np = stamp_all(oo) if payload == "position" else shard_all(oo, make_logical(model, seed, payload, lts=oo.logical_tensors()))
    for key in src_np:                                   # the failed devices' state is lost
        if f[key[0]]:
            src_np[key] = np.full_like(src_np[key], 0xDEAD)
    oo.set_failed(f)
    old, new = E.etc_layout_create(model, old_c), E.etc_layout_create(model, new_c)
    P = max(old.n_dev, new.n_dev)
    ov, need, hold = E.etc_cost_matrix(old, new)
    fd = torch.from_numpy(f).cuda()
    E.etc_mask_failed(ov, hold, fd, old.n_dev)
    o_ov, o_need, o_hold = O.overlap(oo, on)
    assert np.array_equal(ov.cpu().numpy(), o_ov) and np.array_equal(hold.cpu().numpy(), o_hold)
    if device_map is None:
        avail = None
        if avoid_failed:
            a = np.ones(P, np.uint8); a[: old.n_dev][f.astype(bool)] = 0
            if a.sum() >= new.n_dev:
                avail = a
        dm, lb = E.etc_sketch(ov, avail=None if avail is None else torch.from_numpy(avail).cuda())
        ref = O.sketch_hungarian(o_ov, avail)[1]
        assert int(lb.item()) == ref
    else:
        dm = torch.tensor(np.asarray(device_map, np.int32)).cuda()
    dm_h = dm.cpu().numpy()
    plan = E.etc_plan_create(old, new, dm, flags, failed=fd if seed % 2 else f)     # device and host masks
    exp, T, _ = O.migrate(oo, on, dm_h, src_np)
    assert np.array_equal(plan.traffic(), T)
    assert T[: old.n_dev][f.astype(bool)].sum() == 0
    src = upload(src_np)
    dst = E.alloc_buffers(new, fill=0x11)
    stg = torch.empty(max(plan.stats.staging_bytes, 16), dtype=torch.uint8, device="cuda")
    E.etc_migrate(plan, src, dst, stg)
    torch.cuda.synchronize()
    for key, e in exp.items():
        if e.shape[0]:
            assert np.array_equal(download(dst[key], e.itemsize), e), key
    return plan


@pytest.mark.parametrize("name", ["s2", "s4"])
def test_failures_on_scaled_configs(E, name):
    """s2: TP2 PP2 DP2 -> TP4 PP2 DP1 (one replica of each (s,r) may fail); s4: dist-opt old layout — only PARAM is
    replicated there, so any failure is unrecoverable."""
    w = workload(name)
    rng = np.random.default_rng(17)
    if name == "s2":
        for t in range(4):
            f = _survivable_mask(w["old"], rng)
            _run(E, w["model"], w["old"], w["new"], f, 40 + t, flags=t % 2, payload="position" if t == 3 else "stamp")
    else:
        f = np.zeros(16, np.uint8); f[3] = 1
        old, new = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
        with pytest.raises(E.EtcError) as e:
            E.etc_plan_create(old, new, np.arange(32, dtype=np.int32), failed=f)
        assert e.value.code == -8
        oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
        oo.set_failed(f)
        with pytest.raises(O.OracleError) as oe:
            O.migrate(oo, on, np.arange(32, dtype=np.int32), None)
        assert oe.value.code == -8
        E.etc_plan_create(old, new, np.arange(32, dtype=np.int32), failed=np.zeros(16, np.uint8))   # no failure: fine


def test_failures_tiny_sweep(E):
    cfgs = [c for c in tiny_parallel_cfgs(max_devices=8) if not c["dist_opt"]]
    newcfgs = tiny_parallel_cfgs(max_devices=8)
    rng = np.random.default_rng(23)
    ran = 0
    for name, model in tiny_models():
        for t in range(14):
            a = cfgs[rng.integers(len(cfgs))]; b = newcfgs[rng.integers(len(newcfgs))]
            if a["dp"] == 1:
                continue
            try:
                O.Layout(model, a); O.Layout(model, b)
            except O.OracleError:
                continue
            f = _survivable_mask(a, rng)
            na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
            dm = rng.permutation(max(na, nb))[:nb].astype(np.int32) if t % 3 == 0 else None   # may reuse failed slots
            _run(E, model, a, b, f, 500 + t, flags=t % 4 if t % 4 != 2 else 2, device_map=dm)
            ran += 1
    assert ran > 25


def test_all_replicas_failed_is_unrecoverable(E):
    model = dict(tiny_models())["gpt_t"]
    a, b = dict(tp=2, pp=1, dp=2, dist_opt=0), dict(tp=1, pp=1, dp=2, dist_opt=0)
    old, new = E.etc_layout_create(model, a), E.etc_layout_create(model, b)
    f = np.zeros(4, np.uint8); f[1] = f[3] = 1                   # both replicas of tp rank 1
    with pytest.raises(E.EtcError) as e:
        E.etc_plan_create(old, new, np.array([0, 2], np.int32), failed=f)
    assert e.value.code == -8
    f[3] = 0
    E.etc_plan_create(old, new, np.array([0, 2], np.int32), failed=f)


def test_dp_growth_round_robin_balance_on_device(E):
    """PAPER.md:171 (DP growth: counterpart sends its whole state, source groups round-robin): the plan's traffic matrix
    equals the closed form of tests/test_dp_growth_pins.py and the device sketch finds a map that keeps every existing
    group local; s2's model, TP2 PP2, DP 2 -> 5."""
    from test_dp_growth_pins import growth_map, closed_form_T
    from test_gpu_parity import _check_migration
    w = workload("s2")
    old_c, new_c = dict(tp=2, pp=2, dp=2, dist_opt=0), dict(tp=2, pp=2, dp=5, dist_opt=0)
    dm = growth_map(old_c, new_c)
    g = _check_migration(E, w["model"], old_c, new_c, w["seed"], device_map=dm)
    T = g["plan"].traffic()
    assert np.array_equal(T, closed_form_T(old_c, new_c, g["hold"], dm))
    sent = [(int(T[o].sum() - T[o, o]) // int(g["hold"][o])) for o in range(8)]        # whole states sent per old device
    per_group = [sum(sent[o] for o in range(8) if (o // 2) % 2 == d) // 4 for d in range(2)]
    assert sorted(per_group) == [1, 2]                                                   # 3 new groups over 2 old ones
    ov, _, _ = E.etc_cost_matrix(g["old"], g["new"])
    _, lb = E.etc_sketch(ov)
    assert int(lb.item()) == int(g["hold"][:8].sum())


@pytest.mark.parametrize("seed", range(3))
def test_failures_with_every_layout_variant(E, seed):
    """Failure masks on random reconfigurations that draw on every layout variant at once (helpers.random_variant_case):
    the device either reproduces the oracle's result bit for bit or reports the same ETC_ERR_UNRECOVERABLE."""
    from helpers import random_variant_case
    rng = np.random.default_rng(6000 + seed)
    done = unrec = 0
    while done - unrec < 5:                                  # five recoverable cases per seed, plus the unrecoverable ones met on the way
        m, a, b = random_variant_case(rng)
        if a["dp"] < 2:
            continue
        f = _survivable_mask(a, rng)
        if not f.any():
            continue
        na, nb = a["tp"] * a["pp"] * a["dp"], b["tp"] * b["pp"] * b["dp"]
        dm = rng.permutation(max(na, nb))[:nb].astype(np.int32)
        oo, on = O.Layout(m, a), O.Layout(m, b)
        oo.set_failed(f)
        try:
            O.migrate(oo, on, dm, None)
        except O.OracleError as oe:
            assert oe.code == -8
            old, new = E.etc_layout_create(m, a), E.etc_layout_create(m, b)
            with pytest.raises(E.EtcError) as ge:
                E.etc_plan_create(old, new, dm, failed=f)
            assert ge.value.code == -8
            unrec += 1; done += 1
            continue
        _run(E, m, a, b, f, 6100 + done, flags=int(rng.integers(0, 2)), device_map=dm)
        done += 1
    print("unrecoverable cases:", unrec)


def test_dp_isolated_matrix_on_device(E):
    """etc_mask_cross_dp == the oracle's DP-isolated matrix (the paper's formulation, reading A5); on
    config 2 at full size the isolated sketch keeps 2 899 197 952 B local against 5 798 395 904 B for the full matrix
    (SURVEY.md A5 [scratch]); the plan made from the isolated sketch still migrates bit-exactly (s2)."""
    from test_gpu_parity import _check_migration
    w = workload("c2")
    old, new = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    ov, _, _ = E.etc_cost_matrix(old, new)
    assert int(E.etc_sketch(ov)[1].item()) == 5798395904
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    o_iso = O.mask_cross_dp(oo, on, O.overlap(oo, on, method="ranges")[0])
    E.etc_mask_cross_dp(old, new, ov)
    assert np.array_equal(ov.cpu().numpy(), o_iso)
    dm, lb = E.etc_sketch(ov)
    assert int(lb.item()) == 2899197952
    rng = np.random.default_rng(3)
    for name, a, b in [("gpt_t", dict(tp=2, pp=2, dp=2, dist_opt=0), dict(tp=1, pp=2, dp=3, dist_opt=0)),
                       ("llama_u", dict(tp=1, pp=2, dp=4, dist_opt=0), dict(tp=2, pp=2, dp=2, dist_opt=1))]:
        m = dict(tiny_models())[name]
        go, gn = E.etc_layout_create(m, a), E.etc_layout_create(m, b)
        g = E.etc_cost_matrix(go, gn)[0]
        E.etc_mask_cross_dp(go, gn, g)
        lo, ln = O.Layout(m, a), O.Layout(m, b)
        iso = O.mask_cross_dp(lo, ln, O.overlap(lo, ln)[0])
        assert np.array_equal(g.cpu().numpy(), iso)
        dmi, lbi = E.etc_sketch(g)
        assert int(lbi.item()) == O.sketch_hungarian(iso)[1]
        _check_migration(E, m, a, b, 77, device_map=dmi.cpu().numpy())     # the isolated sketch is just another map
