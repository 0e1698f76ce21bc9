"""oracle/defrag.py — TEST INFRASTRUCTURE ONLY.  Plain Python restatement of the paper's virtual rank allocator
(§III-E): Algorithm 2 "Placement-Aware Remapping" and the composition of its migration operators with
the migration sketch (communication coalescing).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.  It
shares no code with paper_2607_04749_b200/ (the CUDA path) and never imports it.

The listing of Algorithm 2 in PAPER.md:226-267 is garbled (1-based `range(1, pw, n)`, `.reversed()` on an iterator,
`cNodes` nested in line 4 but enumerated flat in lines 6-7, `targets` vs `target`); reading A23 restates it from
the prose and this file follows that reading step by step, in the paper's names:

  pw, cw      world size of the prev / curr state;  P = max(pw, cw) physical devices exist (reading A18)
  p2c         pairing from the migration sketch: physical device (= prev process id) -> curr rank;
              here given the other way round as device_map[curr rank] = physical device, as Algorithm 1 returns it
  n           devices per node
  mo          migration operators <a, b>

Pins (tests/test_defrag_pins.py): the two hand-worked examples under tests/golden/ (derived from the prose by hand);
closed forms — after occupancy-level remapping the occupied devices are exactly [0, cw) and no rank already inside
[0, cw) moved, the operator count equals the number of idle devices below cw; after efficiency-level remapping every node
holds exactly its target ranks; composition: coalesced traffic never exceeds two-stage traffic.  "Parity unpinned" with
respect to Fig. 7 (figure absent from PAPER.md).
"""
from __future__ import annotations


def p2c_from_device_map(device_map, P):
    """Invert the sketch: p2c[physical device] = curr rank placed on it, or -1 ("If a process is dropped
    after migration, its id is set to -1")."""
    p2c = [-1] * P
    for rank, dev in enumerate(device_map):
        dev = int(dev)
        if not (0 <= dev < P) or p2c[dev] != -1:
            raise ValueError("device_map is not an injective map into [0, P)")
        p2c[dev] = rank
    return p2c


def defragmentation_for_occupancy(pw, cw, device_map, n):
    """Algorithm 2 lines 1-9 (prose :220).  Returns mo = [(idle device, occupied device), ...]: the
    process on the occupied device moves to the idle device."""
    P = max(pw, cw)
    p2c = p2c_from_device_map(device_map, P)
    # line 3: placement of processes, node by node (n consecutive devices per node)
    pNodes = [list(range(i, min(i + n, P))) for i in range(0, P, n)]
    # line 4: curr rank on every device of every node, -1 = idle
    cNodes = [[p2c[dev] for dev in node] for node in pNodes]
    flat = [x for node in cNodes for x in node]                     # lines 6-7 enumerate devices, not nodes
    # lines 6-7: idle devices in order, occupied devices in reverse order
    idle = [i for i, x in enumerate(flat) if x == -1]
    occu = [i for i, x in enumerate(flat) if x != -1][::-1]
    # lines 8-9: pair them until the two iterators meet
    mo = []
    for i, o in zip(idle, occu):
        if i >= o:                                                  # "are not meeted": the idle slot passed the occupied one
            break
        mo.append((i, o))
    return mo


def defragmentation_for_efficiency(pw, cw, device_map, n):
    """Algorithm 2 lines 10-20 (prose :222).  Returns mo = [(pProc, cProc), ...]: the device that
    should host curr rank pProc (target placement: rank k on device k, so that each TP group sits inside a node) hosts
    cProc (or -1) after the state migration; the operator gives that device the role pProc."""
    P = max(pw, cw)
    p2c = p2c_from_device_map(device_map, P)
    # line 12: optimal placement: curr ranks in order, n per node
    target = [list(range(i, min(i + n, cw))) for i in range(0, cw, n)]
    # lines 14-15: placement after state migration
    devices = [list(range(i, min(i + n, P))) for i in range(0, P, n)]
    loads = [[p2c[dev] for dev in node] for node in devices]
    # line 16: inconsistent node pairs (a node's load is compared on the devices the target uses)
    frag_nodes = [(a, b[:len(a)]) for a, b in zip(target, loads) if a != b[:len(a)]]
    mo = []
    for pNode, cNode in frag_nodes:                                 # lines 17-20
        for pProc, cProc in zip(pNode, cNode):
            if pProc != cProc:
                mo.append((pProc, cProc))
    return mo


def apply_occupancy(device_map, mo):
    """Compose the sketch with occupancy operators (coalescing): the rank that the sketch placed on
    device o is placed on device i instead, in ONE hop from its sources."""
    out = [int(x) for x in device_map]
    where = {dev: rank for rank, dev in enumerate(out)}
    for i, o in mo:
        rank = where.pop(o)
        out[rank] = i
        where[i] = rank
    return out


def apply_efficiency(device_map, mo):
    """Compose the sketch with efficiency operators: curr rank pProc is hosted by device pProc (its target)."""
    out = [int(x) for x in device_map]
    for pProc, _cProc in mo:
        out[pProc] = pProc
    if len(set(out)) != len(out):
        raise ValueError("efficiency remapping produced a non-injective map")
    return out


def defragment(pw, cw, device_map, n, mode):
    """mode: "occupancy" | "efficiency" | "both" (occupancy first, then efficiency on the result).
    Returns (final device_map, number of migration operators emitted)."""
    dm = [int(x) for x in device_map]
    ops = 0
    if mode in ("occupancy", "both"):
        mo = defragmentation_for_occupancy(pw, cw, dm, n)
        dm = apply_occupancy(dm, mo); ops += len(mo)
    if mode in ("efficiency", "both"):
        mo = defragmentation_for_efficiency(pw, cw, dm, n)
        dm = apply_efficiency(dm, mo); ops += len(mo)
    return dm, ops
