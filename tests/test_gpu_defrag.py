"""-m gpu parity of etc_defrag (f1: Algorithm 2 + coalescing) against oracle/defrag.py: operators and
final maps bit-exact; then the composed map through plan + migrate against the element-wise oracle."""
from __future__ import annotations
import os
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from etc_inputs import workload
from oracle import defrag as D
from oracle import oracle as O
from helpers import GOLDEN, make_logical, shard_all, sharded_payload, oracle_migrate


@pytest.fixture(scope="module")
def E():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2607_04749_b200 as E
    E.init()
    return E


MODES = {"occupancy": 1, "efficiency": 2, "both": 3}


def _gpu_defrag(E, dm, pw, cw, n, mode):
    g = torch.tensor(np.asarray(dm, np.int32)).cuda()
    out, n_ops, ops = E.etc_defrag(g, pw, cw, n, MODES[mode])
    out = out.cpu().numpy().tolist(); n_ops = n_ops.cpu().numpy().tolist(); ops = ops.cpu().numpy()
    occ = [tuple(int(v) for v in p) for p in ops[0][: max(n_ops[0], 0)]]
    eff = [tuple(int(v) for v in p) for p in ops[1][: max(n_ops[1], 0)]]
    return out, n_ops, occ, eff


def _oracle_defrag(dm, pw, cw, n, mode):
    dm = [int(x) for x in dm]
    occ, eff = [], []
    if mode in ("occupancy", "both"):
        occ = D.defragmentation_for_occupancy(pw, cw, dm, n)
        dm = D.apply_occupancy(dm, occ)
    if mode in ("efficiency", "both"):
        eff = D.defragmentation_for_efficiency(pw, cw, dm, n)
        dm = D.apply_efficiency(dm, eff)
    return dm, occ, eff


def test_defrag_golden_examples(E):
    """The hand-worked examples (tests/golden/defrag_handworked.txt) through the CUDA kernel."""
    for line in open(os.path.join(GOLDEN, "defrag_handworked.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        head, dm, mo, final = [x.strip() for x in line.split(";")]
        mode, pw, cw, n = head.split()
        ops = [tuple(int(v) for v in t.split(":")) for t in mo.split()]
        out, n_ops, occ, eff = _gpu_defrag(E, [int(x) for x in dm.split()], int(pw), int(cw), int(n), mode)
        assert out == [int(x) for x in final.split()]
        assert (occ if mode == "occupancy" else eff) == ops
        assert n_ops == ([len(ops), 0] if mode == "occupancy" else [0, len(ops)])


def test_defrag_random_maps_vs_oracle(E):
    rng = np.random.default_rng(21)
    shapes = [(8, 4, 4), (16, 12, 4), (12, 5, 2), (32, 8, 8), (9, 9, 3), (4, 8, 4), (64, 48, 8), (1, 1, 1), (5, 1, 8),
              (512, 384, 8), (3000, 2500, 8), (2500, 3000, 4), (1024, 1024, 8), (1025, 1023, 7)]
    for pw, cw, n in shapes:
        P = max(pw, cw)
        for t in range(6 if P < 1000 else 2):
            dm = rng.permutation(P)[:cw]
            if t == 1:
                dm = np.arange(cw)                                   # already compact and at target
            if t == 2:
                dm = np.arange(cw) + (P - cw)                        # everything at the far end
            for mode in MODES:
                out, n_ops, occ, eff = _gpu_defrag(E, dm, pw, cw, n, mode)
                e_out, e_occ, e_eff = _oracle_defrag(dm, pw, cw, n, mode)
                assert out == e_out, (pw, cw, n, mode)
                assert occ == e_occ and eff == e_eff, (pw, cw, n, mode)
                assert n_ops == [len(e_occ), len(e_eff)]


def test_defrag_invalid_maps(E):
    for bad in ([0, 0, 1], [0, 1, 9], [-1, 1, 2]):
        g = torch.tensor(bad, dtype=torch.int32).cuda()
        out, n_ops, _ = E.etc_defrag(g, 4, 3, 2, 3)
        assert (out.cpu().numpy() == -1).all() and (n_ops.cpu().numpy() == -1).all()
    g = torch.tensor([0, 1], dtype=torch.int32).cuda()
    for args in ((0, 2, 2, 3), (2, 2, 0, 3), (2, 2, 2, 0), (2, 2, 2, 4)):
        with pytest.raises(E.EtcError) as e:
            E.etc_defrag(g, *args)
        assert e.value.code == -1


@pytest.mark.parametrize("name,n_per_node", [("s3", 4), ("s2", 4), ("s5", 4)])
@pytest.mark.parametrize("mode", ["occupancy", "both"])
def test_coalesced_migration_vs_oracle(E, name, n_per_node, mode):
    """sketch -> etc_defrag -> plan -> migrate in one hop; the new shards must equal the oracle's element-wise migration
    under the oracle's own composed map, and coalesced traffic <= two-stage traffic."""
    from gpu_helpers import run_gpu_migration
    w = workload(name)
    oo, on = O.Layout(w["model"], w["old"]), O.Layout(w["model"], w["new"])
    old, new = E.etc_layout_create(w["model"], w["old"]), E.etc_layout_create(w["model"], w["new"])
    ov, need, _ = E.etc_cost_matrix(old, new)
    dm, _ = E.etc_sketch(ov)
    final, n_ops, _ = E.etc_defrag(dm, old.n_dev, new.n_dev, n_per_node, MODES[mode])
    dm_h = dm.cpu().numpy()
    e_final, e_occ, e_eff = _oracle_defrag(dm_h, old.n_dev, new.n_dev, n_per_node, mode)
    assert final.cpu().numpy().tolist() == e_final
    src = sharded_payload(oo, w["seed"], "stamp")
    g = run_gpu_migration(w["model"], w["old"], w["new"], src, device_map=np.asarray(e_final, np.int32))
    dst, T, _ = oracle_migrate(oo, on, np.asarray(e_final, np.int32), src)
    assert np.array_equal(g["plan"].traffic(), T)
    for key, exp in dst.items():
        assert np.array_equal(g["dst"][key], exp), key
    if mode == "occupancy":
        # two-stage: the sketch's remote bytes, then every moved rank's whole state once more
        plan0 = E.etc_plan_create(old, new, dm)
        moved = sum(int(need[r].item()) for r in range(new.n_dev) if e_final[r] != int(dm_h[r]))
        assert g["plan"].stats.remote_bytes <= plan0.stats.remote_bytes + moved
