"""paper_2606_15177_b200 -- B200-native (sm_100a) hot path of Gimbal's coordinated MoE
scheduling (arxiv/paper_2606_15177): routing statistics + batched placement objective.

This package is a thin ctypes binding over the C-ABI library `libgimbal.so`
(include/gimbal.h).  It only marshals arguments: every step of the path runs in the CUDA
kernels under csrc/.  PyTorch is used for device memory and streams.  There is no CPU
fallback: loading fails loudly when the library is missing, and the compute calls raise
when no sm_100 device is present.
"""
from .binding import (  # noqa: F401
    GimbalError, RouterCfg, PlacementCfg, StatsState, lib, lib_path, last_error, launch_count,
    route_stats, route_stats_static, STATIC_SCRATCH_BYTES, ABI_VERSION, route_stats_host, eval_placements, eval_placements_host, eval_moves,
    route_stats_workspace_bytes, eval_placements_workspace_bytes, eval_moves_workspace_bytes,
    LOGITS_NONE, LOGITS_OUT, LOGITS_IN, MODE_WINDOW, MODE_EMA, SCORE_SOFTMAX, SCORE_SIGMOID,
    COUNTS_I32, COUNTS_F32, EXPORTED_SYMBOLS, kernel_timing, kernel_elapsed_ms, route_stats_result_bytes,
    KERNEL_ROUTER, KERNEL_GATE, KERNEL_SCORE, KERNEL_MOVES, KERNEL_GREEDY, KERNEL_CHECK, greedy_place, ExpertMap, select_engines,
    order_queues, refine_placement, HostCtx, eval_moves_host, set_option, get_option, ENC_SLOT_TO_EXPERT_I16,
    ENC_EXPERT_TO_RANK_U8, PLACE_TRUSTED, OPT_CTA_GROUP, OPT_FUSE_GATE, OPT_SCORE_GENERIC, OPT_CHECK_SCORES_ALL, OPT_HIST_AGG, OPT_SCORE_TMA, OPT_EPI_PARTS, OPT_PDL, OPT_FUSE_UPDATE,
)
