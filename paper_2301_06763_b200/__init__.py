"""paper_2301_06763_b200 — B200-native hot path of the nested-grid convolution method
(arXiv 2301.06763): libcm (CUDA, sm_100a) behind the C ABI of include/cm.h, plus this
thin ctypes binding.  See DESIGN.md."""
from .binding import (CMError, Plan, cm_debug_copy, cm_green_precompute, cm_plan_create, cm_plan_destroy,
                      cm_plan_kernel_launches, cm_plan_set_G, cm_plan_workspace_bytes, cm_potential,
                      cm_potential_host, cm_potential_profile, cm_acceleration, cm_potential_modified, cm_potential_modified_triplets, cm_direct_sum, cm_slot_to_freq, lib, EXPORTS,
                      cm_plan_prepare_modified, cm_direct_sum_static, cm_direct_sum_static_setup, cm_static_last_error,
                      direct_sum_static, CM_STATIC_MAX_N, cm_shard_restrict, cm_shard_forward, cm_shard_finish,
                      CM_OK, CM_EINVAL, CM_ENOMEM, CM_ECUDA, CM_ENOTREADY,
                      CM_BUF_RESTRICTED, CM_BUF_HOLE, CM_BUF_KHAT)
from ._build import build
from .sharded import LevelShard, LibcmEngine, ShardedSolver, partition_levels

__all__ = [n for n in dir() if not n.startswith("_")]
