"""ctypes binding of include/gimbal.h -- argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))

ABI_VERSION = 300          # GIMBAL_ABI_VERSION of the include/gimbal.h this binding was written against
LOGITS_NONE, LOGITS_OUT, LOGITS_IN = 0, 1, 2
MODE_WINDOW, MODE_EMA = 0, 1
SCORE_SOFTMAX, SCORE_SIGMOID = 0, 1
COUNTS_I32, COUNTS_F32 = 0, 1

EXPORTED_SYMBOLS = [
    "gimbal_version", "gimbal_last_error", "gimbal_launch_count",
    "gimbal_route_stats_workspace_bytes", "gimbal_route_stats", "gimbal_route_stats_static", "gimbal_route_stats_result_bytes",
    "gimbal_route_stats_host", "gimbal_host_ctx_create", "gimbal_host_ctx_destroy", "gimbal_eval_moves_host",
    "gimbal_set_option", "gimbal_get_option",
    "gimbal_eval_placements_workspace_bytes", "gimbal_eval_placements", "gimbal_eval_placements_host",
    "gimbal_eval_moves_workspace_bytes", "gimbal_eval_moves", "gimbal_greedy_place", "gimbal_build_expert_map",
    "gimbal_select_engines", "gimbal_order_queues", "gimbal_refine_placement",
    "gimbal_kernel_timing", "gimbal_kernel_elapsed_ms",
]
KERNEL_ROUTER, KERNEL_GATE, KERNEL_SCORE, KERNEL_MOVES, KERNEL_GREEDY, KERNEL_CHECK = 0, 1, 2, 3, 4, 5
ENC_SLOT_TO_EXPERT_I16, ENC_EXPERT_TO_RANK_U8 = 0, 1
PLACE_TRUSTED = 1
OPT_CTA_GROUP, OPT_FUSE_GATE, OPT_SCORE_GENERIC, OPT_CHECK_SCORES_ALL, OPT_HIST_AGG, OPT_SCORE_TMA, OPT_EPI_PARTS, OPT_PDL, OPT_FUSE_UPDATE = 0, 1, 2, 3, 4, 5, 6, 7, 8


class GimbalError(RuntimeError):
    pass


class _RouterCfg(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("L", "H", "E", "k", "S", "score_fn", "renorm", "n_groups", "topk_groups",
                                          "group_score_topn")] + [("routed_scale", C.c_float)]


class _StatsState(C.Structure):
    _fields_ = [("mode", C.c_int32), ("window_len", C.c_int32), ("ema_decay", C.c_float), ("abi_version", C.c_int32),
                ("A_step", C.c_void_p), ("A_win", C.c_void_p), ("A_pub", C.c_void_p), ("B_pub", C.c_void_p),
                ("A_ema", C.c_void_p), ("B", C.c_void_p), ("pressure_raw", C.c_void_p), ("pressure_rel", C.c_void_p),
                ("step_counter", C.c_void_p), ("status", C.c_void_p)]


class _ExpertMap(C.Structure):
    _fields_ = [("rep_off", C.c_void_p), ("rep_slots", C.c_void_p), ("phys_ids", C.c_void_p), ("NS", C.c_int32)]


class _PlacementCfg(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("L", "E", "G", "slots_per_rank", "S")] + \
               [(n, C.c_float) for n in ("alpha", "beta", "gamma")] + [("counts_dtype", C.c_int32), ("encoding", C.c_int32),
                                                                       ("flags", C.c_int32)]


def lib_path() -> str:
    return os.path.join(_HERE, "libgimbal.so")


_lib = None


def lib():
    """Load libgimbal.so (built in-tree by build.py / __graft_entry__.build()).  No fallback."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise GimbalError(f"{path} is missing: run `python -m paper_2606_15177_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(path)
        L.gimbal_version.restype = C.c_int
        if L.gimbal_version() != ABI_VERSION:
            raise GimbalError(f"{path} has interface version {L.gimbal_version()}, this binding expects {ABI_VERSION}: rebuild it")
        L.gimbal_launch_count.restype = C.c_int64
        for n in ("gimbal_route_stats_workspace_bytes", "gimbal_route_stats_result_bytes",
                  "gimbal_eval_placements_workspace_bytes", "gimbal_eval_moves_workspace_bytes"):
            getattr(L, n).restype = C.c_size_t
        for n in ("gimbal_route_stats", "gimbal_route_stats_static", "gimbal_route_stats_host", "gimbal_eval_placements",
                  "gimbal_eval_placements_host", "gimbal_eval_moves", "gimbal_eval_moves_host", "gimbal_greedy_place",
                  "gimbal_build_expert_map", "gimbal_select_engines", "gimbal_order_queues", "gimbal_refine_placement",
                  "gimbal_host_ctx_create", "gimbal_host_ctx_destroy", "gimbal_set_option", "gimbal_get_option"):
            getattr(L, n).restype = C.c_int
        _lib = L
    return _lib


def last_error() -> str:
    buf = C.create_string_buffer(512)
    lib().gimbal_last_error(buf, C.c_size_t(512))
    return buf.value.decode()


def launch_count() -> int:
    return int(lib().gimbal_launch_count())


def kernel_timing(enable: bool) -> None:
    _check(lib().gimbal_kernel_timing(C.c_int(1 if enable else 0)), "gimbal_kernel_timing")


def kernel_elapsed_ms(which: int) -> float:
    ms = C.c_float(0.0)
    _check(lib().gimbal_kernel_elapsed_ms(C.c_int(which), C.byref(ms)), "gimbal_kernel_elapsed_ms")
    return float(ms.value)


def _check(rc: int, what: str):
    if rc != 0:
        raise GimbalError(f"{what} failed ({rc}): {last_error()}")


def _ptr(t):
    if t is None:
        return C.c_void_p(None)
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous(), "tensors passed to libgimbal must be contiguous"
        return C.c_void_p(t.data_ptr())
    return C.c_void_p(int(t))


def _stream(stream=None):
    if stream is None:
        if not torch.cuda.is_available():      # the library itself reports "no CUDA device"
            return C.c_void_p(None)
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


@dataclass
class RouterCfg:
    L: int
    H: int
    E: int
    k: int
    S: int
    score_fn: int = SCORE_SOFTMAX
    renorm: int = 0
    n_groups: int = 1
    topk_groups: int = 1
    group_score_topn: int = 1
    routed_scale: float = 1.0

    @classmethod
    def from_workload(cls, r):
        return cls(r.L, r.H, r.E, r.k, r.S, r.score_fn, r.renorm, r.n_groups, r.topk_groups, r.group_score_topn,
                   r.routed_scale)

    def c(self):
        return _RouterCfg(self.L, self.H, self.E, self.k, self.S, self.score_fn, self.renorm, self.n_groups,
                          self.topk_groups, self.group_score_topn, self.routed_scale)


@dataclass
class PlacementCfg:
    L: int
    E: int
    G: int
    slots_per_rank: int
    S: int
    alpha: float = 1.0
    beta: float = 0.0025
    gamma: float = 1.0
    counts_dtype: int = COUNTS_I32
    encoding: int = ENC_SLOT_TO_EXPERT_I16
    flags: int = 0

    @property
    def NS(self):
        return self.G * self.slots_per_rank

    def c(self):
        return _PlacementCfg(self.L, self.E, self.G, self.slots_per_rank, self.S, self.alpha, self.beta, self.gamma,
                             self.counts_dtype, self.encoding, self.flags)


class StatsState:
    """Device-resident routing profile (gimbal_stats_state).  Allocation only."""

    def __init__(self, cfg: RouterCfg, mode: int, window_len: int = 1, ema_decay: float = 0.0, device="cuda"):
        L, S, E = cfg.L, cfg.S, cfg.E
        self.cfg, self.mode, self.window_len, self.ema_decay = cfg, mode, window_len, ema_decay
        i32 = dict(dtype=torch.int32, device=device)
        f32 = dict(dtype=torch.float32, device=device)
        self.A_step = torch.zeros(L, S, E, **i32)
        self.A_win = torch.zeros(L, S, E, **i32)
        self.A_pub = torch.zeros(L, S, E, **i32)
        self.B_pub = torch.zeros(L, E, **i32)
        self.A_ema = torch.zeros(L, S, E, **f32)
        self.B = torch.zeros(L, E, **(i32 if mode == MODE_WINDOW else f32))
        self.pressure_raw = torch.zeros(S, **f32)
        self.pressure_rel = torch.zeros(S, **f32)
        self._step_words = torch.zeros(2, dtype=torch.int64, device=device)     # [0] the step index, [1] the library's layer counter
        self.step_counter = self._step_words[:1]
        self.status = torch.zeros(1, **i32)

    @property
    def A_live(self):
        return self.A_win if self.mode == MODE_WINDOW else self.A_ema

    def c(self):
        return _StatsState(self.mode, self.window_len, self.ema_decay, ABI_VERSION, self.A_step.data_ptr(), self.A_win.data_ptr(),
                           self.A_pub.data_ptr(), self.B_pub.data_ptr(), self.A_ema.data_ptr(), self.B.data_ptr(),
                           self.pressure_raw.data_ptr(), self.pressure_rel.data_ptr(), self.step_counter.data_ptr(),
                           self.status.data_ptr())


def route_stats_workspace_bytes(cfg: RouterCfg, n_layers: int, T: int) -> int:
    c = cfg.c()
    return int(lib().gimbal_route_stats_workspace_bytes(C.byref(c), C.c_int(n_layers), C.c_int(T)))


def route_stats(cfg: RouterCfg, state: StatsState, *, T: int, hidden=None, w_router=None, select_bias=None,
                src_logit_bias=None, src_offsets=None, layer0: int = 0, n_layers: int | None = None,
                logits_mode: int = LOGITS_NONE, logits=None, topk_ids=None, topk_w=None, cur_placement=None,
                dp_of_rank=None, G: int = 0, slots_per_rank: int = 0, expert_map=None, phys_ids=None, workspace=None,
                stream=None):
    """gimbal_route_stats (a1..a5).  All tensors are CUDA tensors owned by the caller.
    expert_map = ExpertMap (build_expert_map) + phys_ids [n_layers,T,k] int32: physical slot ids (NEXT-3)."""
    n_layers = cfg.L - layer0 if n_layers is None else n_layers
    c, s = cfg.c(), state.c()
    m = None
    if expert_map is not None:
        m = _ExpertMap(expert_map.rep_off.data_ptr(), expert_map.rep_slots.data_ptr(), phys_ids.data_ptr(), expert_map.NS)
    rc = lib().gimbal_route_stats(C.byref(c), C.c_int(layer0), C.c_int(n_layers), C.c_int(T), _ptr(hidden), _ptr(w_router),
                                  _ptr(select_bias), _ptr(src_logit_bias), _ptr(src_offsets), C.c_int(logits_mode),
                                  _ptr(logits), _ptr(topk_ids), _ptr(topk_w), _ptr(cur_placement), _ptr(dp_of_rank),
                                  C.c_int(G), C.c_int(slots_per_rank), C.byref(s), C.byref(m) if m is not None else C.c_void_p(None),
                                  _ptr(workspace),
                                  C.c_size_t(0 if workspace is None else workspace.numel() * workspace.element_size()),
                                  _stream(stream))
    _check(rc, "gimbal_route_stats")


STATIC_SCRATCH_BYTES = 65536


def route_stats_static(cfg: RouterCfg, state: StatsState, *, T: int, hidden=None, w_router=None, select_bias=None,
                       src_logit_bias=None, src_offsets=None, layer0: int = 0, n_layers: int | None = None,
                       logits_mode: int = LOGITS_NONE, logits=None, topk_ids=None, topk_w=None, cur_placement=None,
                       dp_of_rank=None, G: int = 0, slots_per_rank: int = 0, expert_map=None, phys_ids=None, stream=None):
    """gimbal_route_stats_static: route_stats without a workspace argument, for a caller that cannot obtain device memory
    (an engine that gave all of its HBM to the KV cache, a side thread that must not stall the device with cudaMalloc).
    The update kernel's scratch is a 64 KiB array inside the library, one per GPU and shared by all calls: shapes with
    L * S > 8128 are refused, calls that may overlap on the GPU must be serialised by the caller, and the first call on
    a device (which looks the array up) belongs before any stream capture.  Same results as route_stats."""
    n_layers = cfg.L - layer0 if n_layers is None else n_layers
    c, s = cfg.c(), state.c()
    m = None
    if expert_map is not None:
        m = _ExpertMap(expert_map.rep_off.data_ptr(), expert_map.rep_slots.data_ptr(), phys_ids.data_ptr(), expert_map.NS)
    rc = lib().gimbal_route_stats_static(C.byref(c), C.c_int(layer0), C.c_int(n_layers), C.c_int(T), _ptr(hidden), _ptr(w_router),
                                         _ptr(select_bias), _ptr(src_logit_bias), _ptr(src_offsets), C.c_int(logits_mode),
                                         _ptr(logits), _ptr(topk_ids), _ptr(topk_w), _ptr(cur_placement), _ptr(dp_of_rank),
                                         C.c_int(G), C.c_int(slots_per_rank), C.byref(s),
                                         C.byref(m) if m is not None else C.c_void_p(None), _stream(stream))
    _check(rc, "gimbal_route_stats_static")


class ExpertMap:
    """Device buffers of gimbal_expert_map (allocation + gimbal_build_expert_map)."""

    def __init__(self, L: int, E: int, G: int, slots_per_rank: int, placement, status=None, stream=None):
        self.NS = G * slots_per_rank
        self.rep_off = torch.empty(L, E + 1, dtype=torch.int32, device=placement.device)
        self.rep_slots = torch.empty(L, self.NS, dtype=torch.int16, device=placement.device)
        rc = lib().gimbal_build_expert_map(C.c_int(L), C.c_int(E), C.c_int(G), C.c_int(slots_per_rank), _ptr(placement),
                                           _ptr(self.rep_off), _ptr(self.rep_slots), _ptr(status), _stream(stream))
        _check(rc, "gimbal_build_expert_map")


class HostCtx:
    """gimbal_host_ctx: the copy stream + events of the *_host entry points (one per host thread and device)."""

    def __init__(self):
        self.handle = C.c_void_p(None)
        _check(lib().gimbal_host_ctx_create(C.byref(self.handle)), "gimbal_host_ctx_create")

    def close(self):
        if self.handle:
            lib().gimbal_host_ctx_destroy(self.handle)
            self.handle = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def route_stats_host(ctx: HostCtx, cfg: RouterCfg, state: StatsState, *, T: int, hidden_host, src_offsets_host, hidden_stage,
                     src_offsets_stage, w_router, select_bias=None, src_logit_bias=None, cur_placement=None,
                     dp_of_rank=None, G: int = 0, slots_per_rank: int = 0, result_host=None, workspace=None, stream=None):
    """gimbal_route_stats_host: hidden / src_offsets in (pinned) host memory, results back to host."""
    c, s = cfg.c(), state.c()
    rc = lib().gimbal_route_stats_host(ctx.handle, C.byref(c), C.c_int(T), _ptr(hidden_host), _ptr(src_offsets_host),
                                       _ptr(hidden_stage), C.c_size_t(hidden_stage.numel() * hidden_stage.element_size()),
                                       _ptr(src_offsets_stage), _ptr(w_router), _ptr(select_bias), _ptr(src_logit_bias),
                                       _ptr(cur_placement), _ptr(dp_of_rank), C.c_int(G), C.c_int(slots_per_rank), C.byref(s),
                                       _ptr(result_host), _ptr(workspace),
                                       C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream))
    _check(rc, "gimbal_route_stats_host")


def route_stats_result_bytes(cfg: RouterCfg) -> int:
    c = cfg.c()
    return int(lib().gimbal_route_stats_result_bytes(C.byref(c)))


def eval_placements_workspace_bytes(cfg: PlacementCfg, P: int) -> int:
    c = cfg.c()
    return int(lib().gimbal_eval_placements_workspace_bytes(C.byref(c), C.c_int(P)))


def eval_moves_workspace_bytes(cfg: PlacementCfg) -> int:
    c = cfg.c()
    return int(lib().gimbal_eval_moves_workspace_bytes(C.byref(c)))


def eval_placements(cfg: PlacementCfg, candidates, A, B, D, prev, out, *, M=None, M_scalar: float = 1.0, argmin=None,
                    workspace=None, stream=None):
    """gimbal_eval_placements (a6): out [P,5] = {J, C_load, C_comm, C_mig, maxload}."""
    c = cfg.c()
    P = candidates.shape[0]
    rc = lib().gimbal_eval_placements(C.byref(c), C.c_int(P), _ptr(candidates), _ptr(A), _ptr(B), _ptr(D), _ptr(M),
                                      C.c_float(M_scalar), _ptr(prev), _ptr(out), _ptr(argmin), _ptr(workspace),
                                      C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream))
    _check(rc, "gimbal_eval_placements")


def eval_placements_host(cfg: PlacementCfg, candidates_host, cand_stage, out_stage, A, B, D, prev, out_host, *, M=None,
                         M_scalar: float = 1.0, argmin_host=None, workspace=None, stream=None):
    c = cfg.c()
    P = candidates_host.shape[0]
    rc = lib().gimbal_eval_placements_host(C.byref(c), C.c_int(P), _ptr(candidates_host), _ptr(cand_stage), _ptr(out_stage),
                                           _ptr(A), _ptr(B), _ptr(D), _ptr(M), C.c_float(M_scalar), _ptr(prev),
                                           _ptr(out_host), _ptr(argmin_host), _ptr(workspace),
                                           C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream))
    _check(rc, "gimbal_eval_placements_host")


def eval_moves(cfg: PlacementCfg, cur, prev, A, B, D, delta, *, moves=None, n_moves: int | None = None, M=None,
               M_scalar: float = 1.0, best_per_layer=None, workspace=None, stream=None):
    """gimbal_eval_moves (a7): delta [n,5] = {dJ, dC_load, dC_comm, dC_mig, dmaxload}."""
    c = cfg.c()
    if n_moves is None:
        n_moves = moves.shape[0] if moves is not None else cfg.L * cfg.NS * (cfg.NS - 1) // 2
    rc = lib().gimbal_eval_moves(C.byref(c), _ptr(cur), _ptr(prev), C.c_int64(n_moves), _ptr(moves), _ptr(A), _ptr(B),
                                 _ptr(D), _ptr(M), C.c_float(M_scalar), _ptr(delta), _ptr(best_per_layer), _ptr(workspace),
                                 C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream))
    _check(rc, "gimbal_eval_moves")


def eval_moves_host(cfg: PlacementCfg, cur_host, prev_host, cur_stage, prev_stage, A, B, D, delta_stage, *, moves_host=None,
                    moves_stage=None, n_moves: int | None = None, M=None, M_scalar: float = 1.0, delta_host=None, best_stage=None,
                    best_host=None, workspace=None, stream=None):
    """gimbal_eval_moves_host: cur / prev / moves in host memory; best_host and (optionally) delta_host copied back."""
    c = cfg.c()
    if n_moves is None:
        n_moves = moves_host.shape[0] if moves_host is not None else cfg.L * cfg.NS * (cfg.NS - 1) // 2
    rc = lib().gimbal_eval_moves_host(C.byref(c), _ptr(cur_host), _ptr(prev_host), _ptr(cur_stage), _ptr(prev_stage),
                                      C.c_int64(n_moves), _ptr(moves_host), _ptr(moves_stage), _ptr(A), _ptr(B), _ptr(D), _ptr(M),
                                      C.c_float(M_scalar), _ptr(delta_stage), _ptr(delta_host), _ptr(best_stage), _ptr(best_host),
                                      _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream))
    _check(rc, "gimbal_eval_moves_host")


def set_option(option: int, value: int) -> None:
    _check(lib().gimbal_set_option(C.c_int(option), C.c_int(value)), "gimbal_set_option")


def get_option(option: int) -> int:
    v = C.c_int(0)
    _check(lib().gimbal_get_option(C.c_int(option), C.byref(v)), "gimbal_get_option")
    return int(v.value)


def greedy_place(cfg: PlacementCfg, A, B, D, prev, out, *, M=None, M_scalar: float = 1.0, status=None, stream=None):
    """gimbal_greedy_place (NEXT-1): the paper's online greedy heuristic, out [L,NS] int16 slot -> expert."""
    c = cfg.c()
    rc = lib().gimbal_greedy_place(C.byref(c), _ptr(A), _ptr(B), _ptr(D), _ptr(M), C.c_float(M_scalar), _ptr(prev), _ptr(out),
                                   _ptr(status), _stream(stream))
    _check(rc, "gimbal_greedy_place")


class _SchedCfg(C.Structure):
    _fields_ = [("N", C.c_int32), ("R", C.c_int32)] + [(n, C.c_float) for n in ("high_kv", "large_gap", "lambda_kv", "lambda_moe",
                                                                               "close_frac")]


def select_engines(trace, req_len, comp, rr, engine, *, complete=None, high_kv=0.9, large_gap=0.1, lambda_kv=0.0, lambda_moe=0.0,
                   close_frac=0.0, stream=None):
    """gimbal_select_engines (NEXT-2, Algorithm 1): trace [B,N,4] f32, req_len [B,R] f32, comp [B,N] f64 inout, rr [B] i32
    inout, engine [B,R] i32 out."""
    B, N = trace.shape[0], trace.shape[1]
    R = req_len.shape[1]
    c = _SchedCfg(N, R, high_kv, large_gap, lambda_kv, lambda_moe, close_frac)
    rc = lib().gimbal_select_engines(C.byref(c), C.c_int(B), _ptr(trace), _ptr(complete), _ptr(req_len), _ptr(comp), _ptr(rr),
                                     _ptr(engine), _stream(stream))
    _check(rc, "gimbal_select_engines")


def order_queues(arrival, prefill, qlen, now: float, order, *, theta_age: float = 5.0, stream=None):
    """gimbal_order_queues (Algorithm 2): arrival [B,Q] f32, prefill [B,Q] i32, qlen [B] i32 -> order [B,Q] i32."""
    B, Q = arrival.shape
    rc = lib().gimbal_order_queues(C.c_int(B), C.c_int(Q), _ptr(arrival), _ptr(prefill), _ptr(qlen), C.c_float(now),
                                   C.c_float(theta_age), _ptr(order), _stream(stream))
    _check(rc, "gimbal_order_queues")


def refine_placement(cfg: PlacementCfg, cur, prev, A, B, D, delta, best, *, iters: int = 1, M=None, M_scalar: float = 1.0, applied=None,
                     workspace=None, stream=None):
    """gimbal_refine_placement: `iters` rounds of "apply each layer's best slot exchange"; cur [L,NS] is updated in place."""
    c = cfg.c()
    rc = lib().gimbal_refine_placement(C.byref(c), _ptr(cur), _ptr(prev), C.c_int(iters), _ptr(A), _ptr(B), _ptr(D), _ptr(M),
                                       C.c_float(M_scalar), _ptr(delta), _ptr(best), _ptr(applied), _ptr(workspace),
                                       C.c_size_t(workspace.numel() * workspace.element_size()), _stream(stream))
    _check(rc, "gimbal_refine_placement")
