"""CPU oracle for the Gimbal hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin numpy marshalling around `gimbal_oracle.c` (plain C, fp64; see its header for the
citations, the readings and the pins).  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` leg may import this package.  It imports
nothing from `paper_2606_15177_b200` and shares no code with the CUDA path.

Parity pins: tests/test_oracle_pins.py.  Parity with values printed by the paper is
UNPINNED (the paper prints none for this path; PAPER.md:216-224 holds raw counts only).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gimbal_oracle.c")
_LIB = os.path.join(_HERE, "libgimbal_oracle.so")

SOFTMAX, SIGMOID = 0, 1


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off (sig32 must not be contracted into FMAs)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


class _GateCfg(C.Structure):
    _fields_ = [("E", C.c_int32), ("k", C.c_int32), ("score_fn", C.c_int32), ("renorm", C.c_int32),
                ("n_groups", C.c_int32), ("topk_groups", C.c_int32), ("group_score_topn", C.c_int32),
                ("routed_scale", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_sig32.restype = C.c_float
        _lib.oracle_sig32.argtypes = [C.c_float]
        _lib.oracle_bruteforce.restype = C.c_int64
        _lib.oracle_objective.restype = C.c_int
        _lib.oracle_derived.restype = C.c_int
        _lib.oracle_num_threads.restype = C.c_int
        _lib.oracle_greedy_place.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    """threads of the OpenMP loops (bench.py's single-thread rate); results do not depend on it"""
    lib().oracle_set_num_threads(C.c_int(int(n)))


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def _c(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


# -- a1 ---------------------------------------------------------------------------------
def router_logits(hidden_u16, w_u16, src_logit_bias, src_offsets):
    """hidden_u16 [T,H], w_u16 [E,H] (bf16 bit patterns), src_logit_bias [S,E]|None,
    src_offsets [S+1] -> (logits64 [T,E], logits32 [T,E])."""
    h = _c(hidden_u16, np.uint16); w = _c(w_u16, np.uint16)
    off = _c(src_offsets, np.int32); b = _c(src_logit_bias, np.float32)
    T, H = h.shape; E = w.shape[0]; S = off.shape[0] - 1
    assert w.shape[1] == H
    l64 = np.empty((T, E), np.float64); l32 = np.empty((T, E), np.float32)
    lib().oracle_router_logits(_p(h, C.c_uint16), _p(w, C.c_uint16), _p(b, C.c_float), _p(off, C.c_int32),
                               C.c_int(T), C.c_int(H), C.c_int(E), C.c_int(S), _p(l64, C.c_double), _p(l32, C.c_float))
    return l64, l32


# -- a2 ---------------------------------------------------------------------------------
def sig32(x):
    x = _c(np.atleast_1d(x), np.float32)
    out = np.empty_like(x)
    lib().oracle_sig32_array(_p(x, C.c_float), C.c_int(x.size), _p(out, C.c_float))
    return out


def gate(logits32, rcfg, select_bias=None, tier: int = 1):
    """logits32 [T,E] fp32; rcfg has E,k,score_fn,renorm,n_groups,topk_groups,
    group_score_topn,routed_scale; select_bias [E]|None -> (ids [T,k] int32, w [T,k] f64)."""
    x = _c(logits32, np.float32)
    T, E = x.shape
    assert E == rcfg.E
    cfg = _GateCfg(rcfg.E, rcfg.k, rcfg.score_fn, rcfg.renorm, rcfg.n_groups, rcfg.topk_groups,
                   rcfg.group_score_topn, float(rcfg.routed_scale))
    sb = _c(select_bias, np.float32)
    ids = np.empty((T, rcfg.k), np.int32); w = np.empty((T, rcfg.k), np.float64)
    lib().oracle_gate(C.byref(cfg), _p(x, C.c_float), _p(sb, C.c_float), C.c_int(T), C.c_int(tier),
                      _p(ids, C.c_int32), _p(w, C.c_double))
    return ids, w


# -- a3 ---------------------------------------------------------------------------------
def counts(ids, src_offsets, S: int, E: int):
    ids = _c(ids, np.int32); off = _c(src_offsets, np.int32)
    T, k = ids.shape
    out = np.empty((S, E), np.int64)
    lib().oracle_counts(_p(ids, C.c_int32), _p(off, C.c_int32), C.c_int(T), C.c_int(k), C.c_int(S), C.c_int(E),
                        _p(out, C.c_int64))
    return out


def expert_map(ids, place):
    """ids [T,k] int32 logical experts, place [NS] int16 slot -> expert -> phys [T,k] int32 slots (NEXT-3, R18)."""
    ids = _c(ids, np.int32); place = _c(place, np.int16)
    T, k = ids.shape
    out = np.empty((T, k), np.int32)
    lib().oracle_expert_map(_p(ids, C.c_int32), _p(place, C.c_int16), C.c_int(T), C.c_int(k), C.c_int(place.shape[0]),
                            _p(out, C.c_int32))
    return out


# -- a4 ---------------------------------------------------------------------------------
def update_window(A_win, Cstep, A_pub, step: int, window_len: int) -> bool:
    """in place on int64 arrays; returns True when the window was published."""
    assert A_win.dtype == np.int64 and A_pub.dtype == np.int64 and A_win.flags.c_contiguous and A_pub.flags.c_contiguous
    Cs = _c(Cstep, np.int64)
    pub = C.c_int32(0)
    lib().oracle_update_window(_p(A_win, C.c_int64), _p(Cs, C.c_int64), _p(A_pub, C.c_int64), C.c_int64(A_win.size),
                               C.c_int64(step), C.c_int64(window_len), C.byref(pub))
    return bool(pub.value)


def update_ema(A_ema, Cstep, decay: float) -> None:
    assert A_ema.dtype == np.float64 and A_ema.flags.c_contiguous
    Cs = _c(Cstep, np.int64)
    lib().oracle_update_ema(_p(A_ema, C.c_double), _p(Cs, C.c_int64), C.c_int64(A_ema.size), C.c_double(decay))


# -- a5 ---------------------------------------------------------------------------------
def derived(A, place, dp_of_rank, G: int, sp: int):
    """A [L,S,E]; place [L,NS] int16; -> dict(B [L,E], Lrank [L,G], pressure_raw [S], pressure_rel [S], ok)."""
    A = _c(A, np.float64); place = _c(place, np.int16); dp = _c(dp_of_rank, np.int32)
    L, S, E = A.shape
    B = np.empty((L, E)); Lr = np.empty((L, G)); pr = np.empty(S); pl = np.empty(S)
    ok = lib().oracle_derived(_p(A, C.c_double), _p(place, C.c_int16), _p(dp, C.c_int32), C.c_int(L), C.c_int(S),
                              C.c_int(E), C.c_int(G), C.c_int(sp), _p(B, C.c_double), _p(Lr, C.c_double),
                              _p(pr, C.c_double), _p(pl, C.c_double))
    return dict(B=B, Lrank=Lr, pressure_raw=pr, pressure_rel=pl, ok=bool(ok))


# -- a6 ---------------------------------------------------------------------------------
def _obj_args(A, B, D, M):
    A = _c(A, np.float64); B = _c(B, np.float64); D = _c(D, np.float64); M = _c(M, np.float64)
    return A, B, D, M


def objective(cand, prev, A, B, D, M=None, M_scalar=1.0, *, G, sp, weights=(1.0, 0.0025, 1.0), per_layer=False):
    """cand, prev [L,NS] int16 -> out[5] = {J, C_load, C_comm, C_mig, maxload} (NaN if invalid)."""
    A, B, D, M = _obj_args(A, B, D, M)
    cand = _c(cand, np.int16); prev = _c(prev, np.int16)
    L, S, E = A.shape
    out = np.empty(5); pl = np.empty((L, 4)) if per_layer else None
    lib().oracle_objective(_p(cand, C.c_int16), _p(prev, C.c_int16), _p(A, C.c_double), _p(B, C.c_double),
                           _p(D, C.c_double), _p(M, C.c_double), C.c_double(M_scalar), C.c_int(L), C.c_int(S),
                           C.c_int(E), C.c_int(G), C.c_int(sp), C.c_double(weights[0]), C.c_double(weights[1]),
                           C.c_double(weights[2]), _p(out, C.c_double), _p(pl, C.c_double))
    return (out, pl) if per_layer else out


def objective_batch(cands, prev, A, B, D, M=None, M_scalar=1.0, *, G, sp, weights=(1.0, 0.0025, 1.0)):
    A, B, D, M = _obj_args(A, B, D, M)
    cands = _c(cands, np.int16); prev = _c(prev, np.int16)
    L, S, E = A.shape
    P = cands.shape[0]
    out = np.empty((P, 5))
    lib().oracle_objective_batch(_p(cands, C.c_int16), C.c_int(P), _p(prev, C.c_int16), _p(A, C.c_double),
                                 _p(B, C.c_double), _p(D, C.c_double), _p(M, C.c_double), C.c_double(M_scalar),
                                 C.c_int(L), C.c_int(S), C.c_int(E), C.c_int(G), C.c_int(sp), C.c_double(weights[0]),
                                 C.c_double(weights[1]), C.c_double(weights[2]), _p(out, C.c_double))
    return out


# -- a7 ---------------------------------------------------------------------------------
def all_pair_moves(L: int, NS: int):
    """Canonical order of the implicit neighbourhood: for l, for a < b (a outer, b inner)."""
    a, b = np.triu_indices(NS, 1)
    n = a.size
    mv = np.empty((L, n, 3), np.int32)
    mv[:, :, 0] = np.arange(L)[:, None]
    mv[:, :, 1] = a[None, :]
    mv[:, :, 2] = b[None, :]
    return mv.reshape(-1, 3)


def move_deltas(cur, prev, moves, A, B, D, M=None, M_scalar=1.0, *, G, sp, weights=(1.0, 0.0025, 1.0)):
    """delta [n,5] = {dJ, dC_load, dC_comm, dC_mig, dmaxload} by full re-evaluation."""
    A, B, D, M = _obj_args(A, B, D, M)
    cur = _c(cur, np.int16); prev = _c(prev, np.int16); moves = _c(moves, np.int32)
    L, S, E = A.shape
    n = moves.shape[0]
    out = np.empty((n, 5))
    lib().oracle_move_deltas(_p(cur, C.c_int16), _p(prev, C.c_int16), _p(moves, C.c_int32), C.c_int64(n),
                             _p(A, C.c_double), _p(B, C.c_double), _p(D, C.c_double), _p(M, C.c_double),
                             C.c_double(M_scalar), C.c_int(L), C.c_int(S), C.c_int(E), C.c_int(G), C.c_int(sp),
                             C.c_double(weights[0]), C.c_double(weights[1]), C.c_double(weights[2]), _p(out, C.c_double))
    return out


# -- NEXT-1: greedy heuristic -----------------------------------------------------------
def greedy_place(prev, A, B, D, M=None, M_scalar=1.0, *, G, sp, weights=(1.0, 0.0025, 1.0)):
    """prev [L,NS] int16 -> (ok, placement [L,NS] int16) by the paper's online heuristic."""
    A, B, D, M = _obj_args(A, B, D, M)
    prev = _c(prev, np.int16)
    L, S, E = A.shape
    out = np.empty_like(prev)
    ok = lib().oracle_greedy_place(_p(prev, C.c_int16), _p(A, C.c_double), _p(B, C.c_double), _p(D, C.c_double),
                                   _p(M, C.c_double), C.c_double(M_scalar), C.c_int(L), C.c_int(S), C.c_int(E), C.c_int(G),
                                   C.c_int(sp), C.c_double(weights[0]), C.c_double(weights[1]), C.c_double(weights[2]),
                                   _p(out, C.c_int16))
    return bool(ok), out


# -- NEXT-2: Algorithm 1 ----------------------------------------------------------------
def select_engines(trace, complete, req_len, comp, rr, *, high_kv=0.9, large_gap=0.1, lambda_kv=0.0, lambda_moe=0.0,
                   close_frac=0.0):
    """One scheduler instance: trace [N,4] f32 {kv, pre_rem, wait, moe}, req_len [R] f32, comp [N] f64 (updated in
    place), rr int -> (engine [R] int32, new rr).  PAPER.md:143-167, R19."""
    trace = _c(trace, np.float32); req_len = _c(req_len, np.float32)
    assert comp.dtype == np.float64 and comp.flags.c_contiguous
    N, R = trace.shape[0], req_len.shape[0]
    out = np.empty(R, np.int32); rrv = C.c_int32(int(rr))
    lib().oracle_select_engines(_p(trace, C.c_float), C.c_int(int(bool(complete))), _p(req_len, C.c_float), C.c_int(N), C.c_int(R),
                                C.c_double(high_kv), C.c_double(large_gap), C.c_double(lambda_kv), C.c_double(lambda_moe),
                                C.c_double(close_frac), _p(comp, C.c_double), C.byref(rrv), _p(out, C.c_int32))
    return out, int(rrv.value)


def order_queue(arrival, prefill, now: float, theta_age: float = 5.0):
    """Algorithm 2 (R20): arrival [n] f32 seconds, prefill [n] i32 tokens -> order [n] i32."""
    arrival = _c(arrival, np.float32); prefill = _c(prefill, np.int32)
    out = np.empty(arrival.shape[0], np.int32)
    lib().oracle_order_queue(_p(arrival, C.c_float), _p(prefill, C.c_int32), C.c_int(arrival.shape[0]), C.c_float(now),
                             C.c_float(theta_age), _p(out, C.c_int32))
    return out


def refine(cur, prev, A, B, D, M=None, M_scalar=1.0, *, G, sp, weights=(1.0, 0.0025, 1.0), iters=1):
    """Swap-based local search by full re-evaluation (R21) -> (refined placement [L,NS], applied [L])."""
    A, B, D, M = _obj_args(A, B, D, M)
    cur = np.array(cur, dtype=np.int16, order="C", copy=True); prev = _c(prev, np.int16)
    L, S, E = A.shape
    applied = np.zeros(L, np.int32)
    lib().oracle_refine(_p(cur, C.c_int16), _p(prev, C.c_int16), _p(A, C.c_double), _p(B, C.c_double), _p(D, C.c_double),
                        _p(M, C.c_double), C.c_double(M_scalar), C.c_int(L), C.c_int(S), C.c_int(E), C.c_int(G), C.c_int(sp),
                        C.c_double(weights[0]), C.c_double(weights[1]), C.c_double(weights[2]), C.c_int(iters), _p(applied, C.c_int32))
    return cur, applied


# -- brute force ------------------------------------------------------------------------
def bruteforce(prev, A, B, D, M=None, M_scalar=1.0, *, G, sp, weights=(1.0, 0.0025, 1.0)):
    """One layer, NS == E.  A [S,E], B [E], prev [NS] -> (count, best_J, best_place [NS])."""
    A = _c(A, np.float64); B = _c(B, np.float64); D = _c(D, np.float64); M = _c(M, np.float64)
    prev = _c(prev, np.int16)
    S, E = A.shape
    assert G * sp == E
    bj = C.c_double(0.0); bp = np.empty(E, np.int16)
    n = lib().oracle_bruteforce(_p(prev, C.c_int16), _p(A, C.c_double), _p(B, C.c_double), _p(D, C.c_double),
                                _p(M, C.c_double), C.c_double(M_scalar), C.c_int(S), C.c_int(E), C.c_int(G), C.c_int(sp),
                                C.c_double(weights[0]), C.c_double(weights[1]), C.c_double(weights[2]),
                                C.byref(bj), _p(bp, C.c_int16))
    return int(n), float(bj.value), bp


# -- whole stats step for a set of layers (a1 -> a2 -> a3), the order of PAPER.md:47/212 --
def route_stats_layers(hidden_u16, w_u16, rcfg, src_offsets, src_logit_bias=None, select_bias=None, tier: int = 1):
    """hidden_u16 [n,T,H], w_u16 [n,E,H], src_logit_bias [n,S,E]|None, select_bias [n,E]|None
    -> dict(logits32 [n,T,E], ids [n,T,k], w [n,T,k], C [n,S,E] int64)."""
    n, T, _ = hidden_u16.shape
    S = len(src_offsets) - 1
    out = dict(logits32=np.empty((n, T, rcfg.E), np.float32), ids=np.empty((n, T, rcfg.k), np.int32),
               w=np.empty((n, T, rcfg.k)), C=np.empty((n, S, rcfg.E), np.int64))
    for i in range(n):
        _, l32 = router_logits(hidden_u16[i], w_u16[i], None if src_logit_bias is None else src_logit_bias[i], src_offsets)
        ids, w = gate(l32, rcfg, None if select_bias is None else select_bias[i], tier)
        out["logits32"][i] = l32; out["ids"][i] = ids; out["w"][i] = w
        out["C"][i] = counts(ids, src_offsets, S, rcfg.E)
    return out
