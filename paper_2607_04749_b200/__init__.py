"""paper_2607_04749_b200 — B200-native hot path of ETC's checkpoint-free model-state migration.

Everything computes in the CUDA kernels of libetc.so (include/etc.h); this package is argument marshalling only.
There is no CPU fallback: importing is cheap, but any call raises if libetc.so is missing or no CUDA device exists.
"""
from .binding import (EtcError, Layout, Plan, PlanStats, lib, init,
                      etc_layout_create, etc_cost_matrix, etc_sketch, etc_sketch_static, etc_plan_create, etc_migrate, etc_defrag, etc_mask_failed, etc_plan_set_rounds, etc_migrate_round, RoundInfo,
                      etc_mask_cross_dp, etc_upload_sources, etc_staging_bound, etc_migrate_state, MigrateState,
                      alloc_buffers, kernel_launches,
                      ETC_LOCAL_DIRECT, ETC_ALL_STAGED, ETC_KIND_MAJOR, ETC_ALL_DIRECT, ETC_NO_SYNC, ETC_NO_REORDER, ETC_SKETCH_AUTO, ETC_SKETCH_EXHAUSTIVE, ETC_SKETCH_HUNGARIAN,
                      ETC_PHASE_PACK, ETC_PHASE_UNPACK, ETC_PHASE_ALL, ETC_DEFRAG_OCCUPANCY, ETC_DEFRAG_EFFICIENCY,
                      ETC_DEFRAG_BOTH, ETC_SKETCH_STATIC_MAX_P, ETC_SKETCH_STATIC_SCRATCH_BYTES, EXPORTED_SYMBOLS)
