"""Workload descriptions (plain data, no arithmetic of the method).

The five data configs and the metadata-only config are BASELINE.json `configs`
(model shapes like the paper's GPT-3-style workloads, §IV-A;
reconfigurations like Table II's).  Fields BASELINE.json leaves
open follow DESIGN.md readings A11 (tied embeddings unless "untied" is said),
A13 (max_pos) and the 5b head/ffn/vocab choice.

A workload is a dict:
  {"name", "model": {...}, "old": {"tp","pp","dp","dist_opt"}, "new": {...}, "data": bool}
"""
from __future__ import annotations
import copy
import itertools

KIND_PARAM, KIND_MASTER, KIND_ADAM_M, KIND_ADAM_V = 0, 1, 2, 3
KIND_NAMES = ("param", "master", "adam_m", "adam_v")
STYLE_GPT, STYLE_LLAMA = 0, 1

_ALL4 = 0b1111
_PMV = 0b1101  # PARAM | ADAM_M | ADAM_V (config 1: fp32 params plus Adam m and v, no separate master)


def _model(style, n_layers, hidden, n_q, n_kv, head_dim, ffn, vocab, max_pos, tied, param_bytes, kinds):
    return dict(style=style, n_layers=n_layers, hidden=hidden, n_q_heads=n_q, n_kv_heads=n_kv,
                head_dim=head_dim, ffn_hidden=ffn, vocab=vocab, max_pos=max_pos, tied=tied,
                param_bytes=param_bytes, kinds=kinds)


def _cfg(tp, pp, dp, dist_opt=0):
    return dict(tp=tp, pp=pp, dp=dp, dist_opt=dist_opt)


WORKLOADS = {
    # BASELINE.json configs[0]
    "c1": dict(name="c1", data=True, seed=0xE7C00001,
               model=_model(STYLE_GPT, 2, 256, 4, 4, 64, 1024, 1024, 128, 0, 4, _PMV),
               old=_cfg(2, 2, 1), new=_cfg(1, 2, 2)),
    # BASELINE.json configs[1]
    "c2": dict(name="c2", data=True, seed=0xE7C00002,
               model=_model(STYLE_GPT, 24, 1024, 16, 16, 64, 4096, 50304, 2048, 1, 2, _ALL4),
               old=_cfg(2, 2, 2), new=_cfg(4, 2, 1)),
    # BASELINE.json configs[2]
    "c3": dict(name="c3", data=True, seed=0xE7C00003,
               model=_model(STYLE_GPT, 24, 2048, 32, 32, 64, 8192, 50304, 2048, 1, 2, _ALL4),
               old=_cfg(4, 4, 1), new=_cfg(4, 3, 1)),
    # BASELINE.json configs[3]
    "c4": dict(name="c4", data=True, seed=0xE7C00004,
               model=_model(STYLE_GPT, 32, 2560, 32, 32, 80, 10240, 50304, 2048, 1, 2, _ALL4),
               old=_cfg(2, 4, 2, 1), new=_cfg(4, 2, 4, 1)),
    # BASELINE.json configs[4], data part
    "c5": dict(name="c5", data=True, seed=0xE7C00005,
               model=_model(STYLE_LLAMA, 8, 4096, 32, 8, 128, 14336, 128256, 0, 0, 2, _ALL4),
               old=_cfg(8, 1, 1), new=_cfg(4, 2, 1)),
    # BASELINE.json configs[4], metadata-only part (cost matrix + sketch only)
    "c5b": dict(name="c5b", data=False, seed=0xE7C00006,
                model=_model(STYLE_LLAMA, 80, 8192, 64, 8, 128, 28672, 128256, 0, 0, 2, _ALL4),
                old=_cfg(8, 16, 4), new=_cfg(8, 16, 3)),
    # ---- not BASELINE.json configs: short-row and misaligned stress workloads for the copy kernels.
    # A TP change splits the row-parallel weights (proj, fc2) into column blocks; at high TP degrees the rows of such a
    # slice get short.  c2's model from TP2 PP2 DP2 to TP16: proj slices have rows of 128 B (bf16) / 256 B (fp32).
    "x128": dict(name="x128", data=True, seed=0xE7C00012,
                 model=_model(STYLE_GPT, 24, 1024, 16, 16, 64, 4096, 50304, 2048, 1, 2, _ALL4),
                 old=_cfg(2, 2, 2), new=_cfg(16, 1, 1)),
    # head_dim 32, hidden 512, to TP16: proj rows of 64 B (bf16) / 128 B (fp32), fc2 rows of 256 / 512 B
    "x64": dict(name="x64", data=True, seed=0xE7C00013,
                model=_model(STYLE_GPT, 48, 512, 16, 16, 32, 2048, 50304, 2048, 1, 2, _ALL4),
                old=_cfg(2, 2, 2), new=_cfg(16, 1, 1)),
    # x64 reversed (TP shrinks 16 -> 2): the short rows are on the DESTINATION side (unpack and local copies scatter them)
    "x64r": dict(name="x64r", data=True, seed=0xE7C00015,
                 model=_model(STYLE_GPT, 48, 512, 16, 16, 32, 2048, 50304, 2048, 1, 2, _ALL4),
                 old=_cfg(16, 1, 1), new=_cfg(2, 2, 2)),
    # odd hidden size: every bf16 row is only 2-byte aligned, every fp32 row 4-byte aligned (the re-aligning copy path),
    # c2's reconfiguration
    "xodd": dict(name="xodd", data=True, seed=0xE7C00014,
                 model=_model(STYLE_GPT, 24, 1025, 16, 16, 64, 4096, 50304, 2048, 1, 2, _ALL4),
                 old=_cfg(2, 2, 2), new=_cfg(4, 2, 1)),
}

# Scaled-down twins: same parallel reconfiguration, same style/kinds/tied-ness, dims shrunk so the
# element-wise oracle finishes in seconds while slices still span several copy tiles and ragged tails.
_SCALED = {
    "s2": ("c2", dict(n_layers=4, hidden=192, n_q_heads=12, n_kv_heads=12, head_dim=16, ffn_hidden=768,
                      vocab=3000, max_pos=96)),
    "s3": ("c3", dict(n_layers=12, hidden=256, n_q_heads=8, n_kv_heads=8, head_dim=32, ffn_hidden=1024,
                      vocab=2052, max_pos=64)),
    "s4": ("c4", dict(n_layers=8, hidden=320, n_q_heads=4, n_kv_heads=4, head_dim=80, ffn_hidden=1280,
                      vocab=3004, max_pos=80)),
    "s5": ("c5", dict(n_layers=4, hidden=512, n_q_heads=16, n_kv_heads=8, head_dim=32, ffn_hidden=1792,
                      vocab=4008, max_pos=0)),
    # odd sizes: rows that are not multiples of 16 bytes (exercises the scalar/unaligned copy path)
    "s4odd": ("c4", dict(n_layers=8, hidden=20, n_q_heads=4, n_kv_heads=4, head_dim=5, ffn_hidden=36,
                         vocab=52, max_pos=7)),
    # rows of 388 B (bf16) / 776 B (fp32) at offsets that are only 4- / 8-byte aligned: the re-aligning staged copy path
    "s2odd": ("c2", dict(n_layers=4, hidden=194, n_q_heads=12, n_kv_heads=12, head_dim=16, ffn_hidden=768,
                         vocab=3000, max_pos=96)),
    "s5b": ("c5b", dict(n_layers=16, hidden=64, n_q_heads=16, n_kv_heads=8, head_dim=4, ffn_hidden=128,
                        vocab=256, max_pos=0)),
    # twins of the stress workloads: 16-byte aligned rows of 32 ... 256 B (short-row path), and an odd hidden size
    # (2-byte aligned bf16 rows: the byte-phase re-aligning path)
    "sx64": ("x64", dict(n_layers=4, hidden=256, n_q_heads=16, n_kv_heads=16, head_dim=16, ffn_hidden=1024,
                         vocab=3008, max_pos=64)),
    "sx64r": ("x64r", dict(n_layers=4, hidden=256, n_q_heads=16, n_kv_heads=16, head_dim=16, ffn_hidden=1024,
                           vocab=3008, max_pos=64)),
    "sxodd": ("xodd", dict(n_layers=4, hidden=193, n_q_heads=12, n_kv_heads=12, head_dim=16, ffn_hidden=768,
                           vocab=3000, max_pos=96)),
}


def workload(name: str) -> dict:
    """Return a deep copy of the named workload ("c1".."c5", "c5b", "s2".."s5", "s2odd", "s4odd", "s5b", and the copy-kernel
    stress workloads "x128", "x64", "x64r", "xodd" with their scaled twins "sx64", "sx64r", "sxodd")."""
    if name in WORKLOADS:
        return copy.deepcopy(WORKLOADS[name])
    base, over = _SCALED[name]
    w = copy.deepcopy(WORKLOADS[base])
    w["name"] = name
    w["model"].update(over)
    w["data"] = True
    w["seed"] = WORKLOADS[base]["seed"] ^ 0x5CA1ED
    return w


def scaled_workloads():
    return [workload(k) for k in _SCALED]


def tiny_models():
    """Micro models for exhaustive sweeps (P12): both styles, tied and untied, a non-power-of-two hidden."""
    out = []
    out.append(("gpt_t", _model(STYLE_GPT, 4, 8, 4, 4, 2, 16, 8, 4, 1, 2, _ALL4)))
    out.append(("gpt_u", _model(STYLE_GPT, 2, 24, 4, 4, 6, 20, 12, 3, 0, 4, _PMV)))
    out.append(("gpt_np", _model(STYLE_GPT, 4, 12, 2, 2, 6, 28, 20, 0, 1, 2, _ALL4)))
    out.append(("llama_u", _model(STYLE_LLAMA, 4, 16, 4, 2, 4, 12, 8, 0, 0, 2, _ALL4)))
    out.append(("llama_t", _model(STYLE_LLAMA, 2, 24, 4, 4, 6, 20, 16, 0, 1, 2, _ALL4)))
    return out


def tiny_parallel_cfgs(max_devices=8, sizes=(1, 2, 4)):
    """All (tp,pp,dp,dist_opt) with sizes in `sizes` and tp*pp*dp <= max_devices."""
    out = []
    for tp, pp, dp in itertools.product(sizes, sizes, sizes):
        if tp * pp * dp <= max_devices:
            out.append(_cfg(tp, pp, dp, 0))
            if dp > 1:
                out.append(_cfg(tp, pp, dp, 1))
    return out
