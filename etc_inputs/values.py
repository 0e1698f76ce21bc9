"""Seeded, counter-based value generators (no layout logic, no arithmetic of the method).

`logical_values` produces the values of one LOGICAL tensor (kind, tensor id, element count): the
caller (a test, through the oracle) decides how they are sharded.  Distributions follow
BASELINE.json `configs`: params/master ~ N(0, 0.02), Adam m ~ N(0, 1e-3), Adam v ~ U[0, 1e-4);
bf16 params are the round-to-nearest-even of the fp32 master value (reading A15).

`index_stamp` / `position_stamp` are the certain-detection payloads of pins P8 / P9.
"""
from __future__ import annotations
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
    z = x
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
    return z ^ (z >> np.uint64(31))


def _counter(seed: int, stream: int, tensor_id: int, n: int) -> np.ndarray:
    base = (np.uint64(seed & 0xFFFFFFFF) << np.uint64(32)) ^ (np.uint64(stream) << np.uint64(24)) \
        ^ np.uint64(tensor_id & 0xFFFFFF)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.array([base], dtype=np.uint64))[0]
        return _splitmix64(np.arange(n, dtype=np.uint64) * np.uint64(0xD1342543DE82EF95) + key)


def _normal(seed, stream, tensor_id, n, std):
    h = _counter(seed, stream, tensor_id, n)
    u1 = ((h >> np.uint64(40)).astype(np.float64) + 1.0) / 16777217.0      # (0,1)
    u2 = ((h & np.uint64(0xFFFFFF)).astype(np.float64)) / 16777216.0        # [0,1)
    z = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return (z * std).astype(np.float32)


def _uniform(seed, stream, tensor_id, n, hi):
    h = _counter(seed, stream, tensor_id, n)
    u = (h >> np.uint64(40)).astype(np.float64) / 16777216.0
    return (u * hi).astype(np.float32)


def fp32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns."""
    b = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((b >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((b + r) >> np.uint32(16)).astype(np.uint16)


def logical_values(seed: int, kind: int, tensor_id: int, n: int, elem_bytes: int) -> np.ndarray:
    """Values of one logical tensor of one state kind, as raw little-endian words.

    Returns uint16 (elem_bytes == 2, bf16 bit patterns) or uint32 (elem_bytes == 4, fp32 bit patterns).
    kind: 0 PARAM, 1 MASTER, 2 ADAM_M, 3 ADAM_V.  PARAM and MASTER draw from the same stream, so the bf16
    param equals RNE(master) element by element.
    """
    if kind in (0, 1):
        v = _normal(seed, 1, tensor_id, n, 0.02)
    elif kind == 2:
        v = _normal(seed, 2, tensor_id, n, 1e-3)
    elif kind == 3:
        v = _uniform(seed, 3, tensor_id, n, 1e-4)
    else:
        raise ValueError(kind)
    if elem_bytes == 2:
        return fp32_to_bf16_bits(v)
    if elem_bytes == 4:
        return v.view(np.uint32).copy()
    raise ValueError(elem_bytes)


def index_stamp(kind: int, tensor_id: int, n: int, elem_bytes: int, salt: int = 0) -> np.ndarray:
    """P8: a hash of (kind, tensor, flat index) per logical element: any misplaced element differs.  `salt` gives a
    different (equally cheap) payload of the same kind, for tests that push several payloads through one plan."""
    with np.errstate(over="ignore"):
        h = _splitmix64(np.arange(n, dtype=np.uint64) + (np.uint64(kind) << np.uint64(56))
                        + (np.uint64(tensor_id) << np.uint64(36)) + np.uint64(salt & 0xFFFFFFFF) * np.uint64(0x9E3779B97F4A7C15))
    if elem_bytes == 2:
        return (h & np.uint64(0xFFFF)).astype(np.uint16)
    return (h & np.uint64(0xFFFFFFFF)).astype(np.uint32)


def _pos_words(dev: int, kind: int, idx):
    # layout-agnostic: depends only on which buffer (dev, kind) and the position inside it
    return (idx * 2654435761 + dev * 40503 + kind * 9176 + 12345)


def position_stamp(dev: int, kind: int, n: int, elem_bytes: int, start: int = 0) -> np.ndarray:
    """P9: every element of buffer (dev, kind) carries a function of (dev, kind, position) only."""
    idx = np.arange(start, start + n, dtype=np.uint64)
    w = _pos_words(dev, kind, idx)
    if elem_bytes == 2:
        return ((w >> np.uint64(7)) & np.uint64(0xFFFF)).astype(np.uint16)
    return ((w >> np.uint64(5)) & np.uint64(0xFFFFFFFF)).astype(np.uint32)


def position_stamp_at(dev: int, kind: int, idx, elem_bytes: int) -> np.ndarray:
    """`position_stamp` evaluated at arbitrary positions idx (int array)."""
    w = _pos_words(dev, kind, np.asarray(idx).astype(np.uint64))
    if elem_bytes == 2:
        return ((w >> np.uint64(7)) & np.uint64(0xFFFF)).astype(np.uint16)
    return ((w >> np.uint64(5)) & np.uint64(0xFFFFFFFF)).astype(np.uint32)


def position_stamp_torch(dev: int, kind: int, n: int, elem_bytes: int, device):
    """Same values as `position_stamp`, produced directly in device memory (int16 / int32 bit patterns)."""
    import torch
    out = torch.empty(n, dtype=torch.int16 if elem_bytes == 2 else torch.int32, device=device)
    step = 1 << 24
    for s in range(0, n, step):
        m = min(step, n - s)
        idx = torch.arange(s, s + m, dtype=torch.int64, device=device)
        w = idx * 2654435761 + (dev * 40503 + kind * 9176 + 12345)
        if elem_bytes == 2:
            out[s:s + m] = ((w >> 7) & 0xFFFF).to(torch.int16)
        else:
            out[s:s + m] = ((w >> 5) & 0xFFFFFFFF).to(torch.int32)
    return out


def bench_fill_torch(buf, kind: int, seed: int):
    """Fill a device buffer (bf16 or fp32 tensor) in place with the workload's value distribution.

    Used by bench.py for full-size configs: timing does not depend on replica consistency, so the buffer is
    filled directly instead of being sharded from logical tensors on the host.
    """
    import torch
    g = torch.Generator(device=buf.device)
    g.manual_seed(seed)
    step = 1 << 26
    flat = buf.view(-1)
    for s in range(0, flat.numel(), step):
        part = flat[s:s + step]
        if kind in (0, 1):
            part.normal_(0.0, 0.02, generator=g)
        elif kind == 2:
            part.normal_(0.0, 1e-3, generator=g)
        else:
            part.uniform_(0.0, 1e-4, generator=g)
    return buf
