"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds ONLY workload descriptions (plain data) and seeded value
generators.  It contains none of the method's arithmetic: no layout rule, no
index map, no cost/overlap/sketch/plan logic.  Neither `oracle/` nor
`paper_2607_04749_b200/` is imported from here.
"""
from .workloads import (KIND_PARAM, KIND_MASTER, KIND_ADAM_M, KIND_ADAM_V, KIND_NAMES,
                        STYLE_GPT, STYLE_LLAMA, WORKLOADS, workload, scaled_workloads,
                        tiny_models, tiny_parallel_cfgs)
from .values import (logical_values, index_stamp, position_stamp, position_stamp_at, position_stamp_torch,
                     fp32_to_bf16_bits, bench_fill_torch)
