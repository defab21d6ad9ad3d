#!/usr/bin/env python
"""bench.py -- one JSON line for the Gimbal hot path on B200.

A "step" is one pass of the whole hot path over one batch of synthetic input:
  gimbal_route_stats     a1-a5  router GEMM + gating + [L,S,E] histogram + window/EMA + load/pressure
  gimbal_eval_placements a6     P candidate placements scored against the live profile
  gimbal_eval_moves      a7     the whole single-move neighbourhood of the current placement
`value` = routed tokens/s = T / (device time of one step), inputs resident in HBM.
`e2e`   = the same metric through the *_host C-ABI calls: hidden states, source offsets and the
          candidates start in pinned HOST memory each step and the results are read back.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload v3] [--impl reference]

N > 1 (under torch.distributed.run): the path has no cross-GPU exchange (north_star: EP ranks
and DP engines are logical partitions on one GPU), so every rank runs an independent replica
of the step ("replicas only", weak scaling) and `value` adds the ranks up.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import gen, get_workload, scaled  # noqa: E402
from workloads.configs import MODE_WINDOW  # noqa: E402

METRIC = "routed tokens/s (stats path + placement scoring, whole hot path)"
# dram__bytes_read + dram__bytes_write of router_gemm_kernel per token-layer at the V3 shape, from the committed
# `ncu --set full` capture profiles/r1_ncu_k1_router_gemm.txt: (5.661509e9 + 3.763712e6) B over 65536 tokens x 6 layers
# (algorithmic: 2*H = 14336 B).  The capture covers 6 of the 58 layers; traffic per launch scales it by T*L.
# smsp__inst_executed.sum of place_score_fast_kernel<9,32,1,0> per (candidate, layer) at the V3 shape, from
# profiles/r1_ncu_k4_k5_placement.txt (46,644,992 warp instructions for 4096 x 58 units): the kernel is issue-bound, so
# its ALU roofline (148 SMs x 4 schedulers x 1 warp instruction per clock at the maximum SM clock)
# is reported next to the HBM one.
NCU_WARP_INSTR_PER_UNIT_K4_V3 = 46644992 / (4096 * 58)
NCU_DRAM_BYTES_PER_TOKEN_LAYER_V3 = (5.661509e9 + 3.763712e6) / (65536 * 6)


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm=p["hbm_gbs"], tf_burst=p["bf16_tflops"], tf_sustained=p.get("bf16_tflops_sustained", p["bf16_tflops"]),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sustained=1400.0, source="fallback (B200_PROFILING.md)")


# --------------------------------------------------------------------------------------------
# clocks during the timed region
# --------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.proc, self.path = gpu_index, None, f"/tmp/gimbal_clocks_{os.getpid()}.csv"

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                                          "-i", str(self.gpu)], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[])
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for line in open(self.path):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            try:
                pw.append(float(f[3]))
            except ValueError:
                pass
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if sm:
            busy = [x for x in sm if x > 0]
            out.update(sm_mhz=statistics.median(busy or sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=(max(pw) if pw else None))
        return out


# --------------------------------------------------------------------------------------------
# oracle timing (cpu_baseline / --impl reference)
# --------------------------------------------------------------------------------------------
def oracle_step_time(w, sample_tokens, sample_layers, sample_P, sample_moves, place_layers=None):
    """Times the CPU oracle, as it stands, on a bounded sample of the workload and extrapolates
    to one full step.  Returns (seconds per full step, description, threads)."""
    import oracle
    r = w.router
    ws = scaled(w, L=sample_layers, T=sample_tokens)
    hidden = gen.hidden_all(ws, 0, "cpu")
    W = gen.w_router(ws, "cpu")
    slb = gen.src_logit_bias(ws, 0, "cpu").numpy()
    sb = gen.select_bias(ws, "cpu")
    off = gen.src_offsets(ws, 0, sample_tokens, "cpu").numpy()
    hb = hidden.view(torch.int16).numpy().view(np.uint16)
    wb = W.view(torch.int16).numpy().view(np.uint16)
    t0 = time.perf_counter()
    res = oracle.route_stats_layers(hb, wb, r, off, slb, None if sb is None else sb.numpy(), tier=1)
    A = np.zeros((sample_layers, r.S, r.E)); oracle.update_ema(A, res["C"], 0.9)
    t_stats = time.perf_counter() - t0
    tok_layers_per_s = sample_tokens * sample_layers / t_stats
    # placement side on a profile of the right shape
    place_layers = sample_layers if place_layers is None else place_layers
    A_full = np.repeat(res["C"][:1], place_layers, 0).astype(np.float64)
    B_full = A_full.sum(1)
    wl = scaled(w, L=place_layers, P=sample_P)
    prev = gen.prev_placement(wl, B_full, "cpu")
    cands = gen.candidates(wl, prev, sample_P, "cpu").numpy()
    D = gen.comm_cost_D(wl, "binary", "cpu").numpy()
    dp = gen.dp_of_rank(wl, "cpu").numpy()
    t0 = time.perf_counter()
    oracle.derived(A_full, prev.numpy(), dp, w.G, w.slots_per_rank)
    oracle.objective_batch(cands, prev.numpy(), A_full, B_full, D, None, 1.0, G=w.G, sp=w.slots_per_rank)
    t_obj = time.perf_counter() - t0
    cand_layers_per_s = sample_P * place_layers / t_obj
    moves = gen.explicit_moves(wl, sample_moves, "cpu").numpy()
    t0 = time.perf_counter()
    oracle.move_deltas(prev.numpy(), prev.numpy(), moves, A_full, B_full, D, None, 1.0, G=w.G, sp=w.slots_per_rank)
    t_mv = time.perf_counter() - t0
    moves_per_s = sample_moves / t_mv
    n_moves = r.L * w.NS * (w.NS - 1) // 2
    step_s = w.T * r.L / tok_layers_per_s + w.P * r.L / cand_layers_per_s + n_moves / moves_per_s
    desc = (f"oracle as it stands: a1-a5 on {sample_tokens} tokens x {sample_layers} layers ({t_stats:.1f}s, "
            f"{tok_layers_per_s:.0f} token-layers/s), a6 on {sample_P} candidates x {place_layers} layers ({t_obj:.1f}s, "
            f"{cand_layers_per_s:.0f} candidate-layers/s), a7 on {sample_moves} moves ({t_mv:.1f}s, {moves_per_s:.0f} moves/s); "
            f"extrapolated to one full step (T={w.T}, L={r.L}, P={w.P}, {n_moves} moves)")
    return step_s, desc, oracle.num_threads(), dict(token_layers_per_s=tok_layers_per_s, candidate_layers_per_s=cand_layers_per_s,
                                                     moves_per_s=moves_per_s)


SAMPLES = {   # workload -> (tokens, layers, candidates, moves, placement layers) of the oracle sample (~10-30 s of CPU work)
    "tiny": (4096, 1, 64, 120, 1), "v2lite": (16384, 26, 1024, 100000, 26), "qwen3": (32768, 8, 512, 100000, 48),
    "v3": (16384, 4, 1024, 100000, 58), "decode": (256, 58, 1024, 100000, 58),
}


def _sample(w, scale: float = 1.0):
    """scale < 1 shrinks the sample (reference arm: K + W samples must end within a few minutes)."""
    tok, lay, P, mv, pl = SAMPLES[w.name]
    tok, P, mv = max(256, int(tok * scale)), max(16, int(P * scale)), max(120, int(mv * scale))
    return min(tok, w.T), min(lay, w.router.L), min(P, w.P), mv, min(pl, w.router.L)


# --------------------------------------------------------------------------------------------
# N > 1: independent replicas; the only cross-rank step is the max of the timings
# --------------------------------------------------------------------------------------------
def max_over_ranks(ms: float, device="cpu") -> float:
    """Slowest rank's time (torch.distributed must be initialised; works on gloo and nccl)."""
    import torch.distributed as td
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    td.all_reduce(t, op=td.ReduceOp.MAX)
    return float(t.item())


def replica_value(tokens_per_rank: int, world: int, ms_per_step: float) -> float:
    """Whole-job routed tokens/s of `world` replicas that each process tokens_per_rank per step."""
    return world * tokens_per_rank / (ms_per_step * 1e-3)


# --------------------------------------------------------------------------------------------
def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    times, desc, threads = [], "", 1
    scale = min(1.0, 8.0 / (args.warmup + args.steps))         # a full sample is ~15 s; keep the whole run near 2 minutes
    for i in range(args.warmup + args.steps):
        s, desc, threads, _ = oracle_step_time(w, *_sample(w, scale))
        if i >= args.warmup:
            times.append(s)
    step_s = sum(times) / len(times)
    value = w.T / step_s
    cb = dict(value=value, unit="routed tokens/s", cores=threads, kind="oracle", sample=desc)
    line = dict(impl="reference", metric=METRIC, value=value, unit="routed tokens/s", n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=step_s * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=_config(w, args), cpu_baseline=cb,
                e2e=dict(value=value, unit="routed tokens/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


def _config(w, args):
    r = w.router
    return dict(workload=f"{w.name}: L={r.L} H={r.H} E={r.E} top-{r.k} S={r.S} T={w.T}/step; G={w.G}x{w.slots_per_rank} slots, P={w.P}, "
                         f"full move neighbourhood ({r.L * w.NS * (w.NS - 1) // 2} moves)",
                parallelism="replicas only (no cross-GPU exchange on this path)",
                l2="hidden states of one step (>> L2) stream through L2 between the placement kernels; an explicit 256 MiB flush runs "
                   "between timed steps, outside the timed events",
                outputs="A_step/B/pressure (a3-a5), out[P,5]+argmin (a6), delta[n,5]+best_per_layer (a7); top-k ids and weights "
                        + ("written" if getattr(args, "with_ids", False) else "not written"))


def run_ours(args, w):
    import paper_2606_15177_b200 as g

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = world > 1
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if dist:
        import torch.distributed as td
        td.init_process_group("nccl")
    if not os.path.exists(g.lib_path()):
        raise SystemExit("libgimbal.so missing: run __graft_entry__.build() -- there is no CPU fallback")
    peaks = _peaks()
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    torch.manual_seed(1234 + rank)

    # ---- inputs, resident in HBM -------------------------------------------------------------
    hidden = gen.hidden_all(w, rank, dev)                      # [L,T,H] bf16, distinct per layer (and per rank)
    W = gen.w_router(w, dev)
    slb = gen.src_logit_bias(w, 0, dev)
    sb = gen.select_bias(w, dev)
    off = gen.src_offsets(w, 0, w.T, dev)
    dp = gen.dp_of_rank(w, dev)
    D = gen.comm_cost_D(w, "binary", dev)
    st = g.StatsState(cfg, w.mode, window_len=max(w.window_len, 1), ema_decay=w.ema_decay, device=dev)
    ws_r = torch.empty(g.route_stats_workspace_bytes(cfg, r.L, w.T), dtype=torch.uint8, device=dev)
    pc = g.PlacementCfg(L=r.L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S,
                        counts_dtype=g.COUNTS_I32 if w.mode == MODE_WINDOW else g.COUNTS_F32)
    # one un-timed stats step gives the profile the placement side starts from
    g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off, workspace=ws_r)
    torch.cuda.synchronize()
    prev = gen.prev_placement(w, st.B.cpu().numpy(), dev)
    cands = gen.candidates(w, prev, w.P, dev)
    cur = cands[min(2, w.P - 1)].contiguous()
    n_moves = r.L * w.NS * (w.NS - 1) // 2
    out = torch.empty(w.P, 5, device=dev)
    argmin = torch.zeros(1, dtype=torch.int32, device=dev)
    delta = torch.empty(n_moves, 5, device=dev)
    best = torch.zeros(r.L, dtype=torch.int32, device=dev)
    ws_p = torch.empty(g.eval_placements_workspace_bytes(pc, w.P), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    # profile the placement side reads: this step's counts (window mode) or the EMA state
    A_live, B_live = (st.A_step if w.mode == MODE_WINDOW else st.A_ema), st.B

    ids_out = torch.empty(r.L, w.T, r.k, dtype=torch.int32, device=dev) if args.with_ids else None
    w_out = torch.empty(r.L, w.T, r.k, dtype=torch.float32, device=dev) if args.with_ids else None

    def step():
        g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                      topk_ids=ids_out, topk_w=w_out,
                      cur_placement=cur, dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws_r)
        g.eval_placements(pc, cands, A_live, B_live, D, prev, out, argmin=argmin, workspace=ws_p)
        g.eval_moves(pc, cur, prev, A_live, B_live, D, delta, best_per_layer=best, workspace=ws_p)

    g.kernel_timing(True)
    # NEXT-1 (not part of the timed step): the greedy heuristic on the same profile, timed on its own
    greedy_out = torch.empty_like(prev)
    greedy_ms = []
    for _ in range(4):
        g.greedy_place(pc, A_live, B_live, D, prev, greedy_out)
        greedy_ms.append(g.kernel_elapsed_ms(g.KERNEL_GREEDY))
    # K2 (not part of the timed step): the standalone gating + histogram kernel on given logits (LOGITS_IN), the
    # kernel whose roofline is plain HBM: 4*E bytes read per token-layer.  Logits of `nl` layers (> L2) are
    # written once by the fused kernel's LOGITS_OUT mode, then re-read from HBM.
    nl = min(r.L, max(1, (768 << 20) // (w.T * r.E * 4)))
    lg = torch.empty(nl, w.T, r.E, device=dev)
    st2 = g.StatsState(g.RouterCfg(nl, r.H, r.E, r.k, r.S, r.score_fn, r.renorm, r.n_groups, r.topk_groups, r.group_score_topn,
                                   r.routed_scale), w.mode, window_len=1, ema_decay=w.ema_decay, device=dev)
    g.route_stats(st2.cfg, st2, T=w.T, hidden=hidden[:nl], w_router=W[:nl], select_bias=None if sb is None else sb[:nl],
                  src_logit_bias=slb[:nl], src_offsets=off, logits_mode=g.LOGITS_OUT, logits=lg, workspace=ws_r)
    gate_ms = []
    for _ in range(4):
        flush.zero_()
        g.route_stats(st2.cfg, st2, T=w.T, select_bias=None if sb is None else sb[:nl], src_offsets=off, logits_mode=g.LOGITS_IN,
                      logits=lg, workspace=ws_r)
        gate_ms.append(g.kernel_elapsed_ms(g.KERNEL_GATE))
    del lg
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    # ---- timed region: K steps, CUDA events per step on the launching stream, L2 flushed in between ----
    sampler = ClockSampler(local)
    if dist:
        td.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    k_router, k_score, k_moves = [], [], []
    launches0 = g.launch_count()
    for s0, s1 in ev:
        flush.zero_()
        s0.record()
        step()
        s1.record()
        k_router.append(g.kernel_elapsed_ms(g.KERNEL_ROUTER))
        k_score.append(g.kernel_elapsed_ms(g.KERNEL_SCORE))
        k_moves.append(g.kernel_elapsed_ms(g.KERNEL_MOVES))
    torch.cuda.synchronize()
    launches = g.launch_count() - launches0
    if dist:
        td.barrier()
    clocks = sampler.stop()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    if dist:
        total_ms = max_over_ranks(total_ms, dev)
    ms_per_step = total_ms / args.steps
    value = replica_value(w.T, world, ms_per_step)

    # ---- roofline of the dominant kernel (router GEMM with fused gating + histogram) -------------------
    gemm_ms = statistics.mean(k_router)
    flops = 2.0 * w.T * r.H * r.E * r.L                       # 2*H*E flop per token-layer
    bytes_hidden = 2.0 * w.T * r.H * r.L                      # 2*H bytes per token-layer, read exactly once
    tf = flops / (gemm_ms * 1e-3) / 1e12
    roofline = dict(bound="tensor", achieved=tf, peak=peaks["tf_sustained"], unit="TFLOP/s", frac=tf / peaks["tf_sustained"],
                    traffic=(NCU_DRAM_BYTES_PER_TOKEN_LAYER_V3 * w.T * r.L if w.name == "v3" else None),
                    traffic_unit="bytes per launch (ncu dram read+write per token-layer x T x L, profiles/r1_ncu_k1_router_gemm.txt)",
                    algorithmic_bytes=bytes_hidden, algorithmic_flops=flops,
                    kernel="router_gemm_kernel (a1 + fused a2/a3)", ms=gemm_ms, share_of_step=gemm_ms / ms_per_step,
                    peak_source=peaks["source"] + ", sustained bf16 (kernel timed inside a long step)",
                    frac_of_burst_peak=tf / peaks["tf_burst"],
                    hbm=dict(achieved=bytes_hidden / (gemm_ms * 1e-3) / 1e9, peak=peaks["hbm"], unit="GB/s",
                             frac=bytes_hidden / (gemm_ms * 1e-3) / 1e9 / peaks["hbm"],
                             note="same kernel against the HBM roofline: 2*H bytes of hidden per token-layer"))
    score_ms, moves_ms = statistics.mean(k_score), statistics.mean(k_moves)
    cand_bytes = 2.0 * r.L * w.NS * w.P
    gate_bytes = 4.0 * r.E * w.T * nl
    extra = dict(
        gate_hist_kernel=dict(ms=min(gate_ms[1:]), layers=nl, bound="hbm", achieved=gate_bytes / (min(gate_ms[1:]) * 1e-3) / 1e9,
                              peak=peaks["hbm"], unit="GB/s", frac=gate_bytes / (min(gate_ms[1:]) * 1e-3) / 1e9 / peaks["hbm"],
                              algorithmic_bytes="4*E per token-layer (logits read once; counts only)",
                              note="a2+a3 standalone on given logits (LOGITS_IN); outside the timed step"),
        greedy_place_kernel=dict(ms=min(greedy_ms[1:]), layers=r.L, note="NEXT-1, PAPER.md:260-268; outside the timed step"),
        placements_per_s=world * w.P / (score_ms * 1e-3), moves_per_s=world * n_moves / (moves_ms * 1e-3),
        place_score_kernel=dict(ms=score_ms, bound="hbm", achieved=cand_bytes / (score_ms * 1e-3) / 1e9, peak=peaks["hbm"],
                                unit="GB/s", frac=cand_bytes / (score_ms * 1e-3) / 1e9 / peaks["hbm"],
                                algorithmic_bytes="2*L*NS per candidate",
                                alu=(dict(achieved=NCU_WARP_INSTR_PER_UNIT_K4_V3 * w.P * r.L / (score_ms * 1e-3) / 1e9,
                                          peak=148 * 4 * 1.965, unit="G warp-instructions/s",
                                          frac=NCU_WARP_INSTR_PER_UNIT_K4_V3 * w.P * r.L / (score_ms * 1e-3) / 1e9 / (148 * 4 * 1.965),
                                          note="issue-bound kernel: instructions per unit from the committed ncu capture; peak at "
                                               "the maximum SM clock (1965 MHz)") if w.name == "v3" else None)),
        move_delta_kernel=dict(ms=moves_ms, bound="hbm", achieved=20.0 * n_moves / (moves_ms * 1e-3) / 1e9, peak=peaks["hbm"],
                               unit="GB/s", frac=20.0 * n_moves / (moves_ms * 1e-3) / 1e9 / peaks["hbm"],
                               algorithmic_bytes="20 B written per move (implicit neighbourhood)"))

    # ---- e2e: the same step through the *_host entry points ------------------------------------------
    e2e = None
    import psutil
    fits = hidden.numel() * 2 * world < 0.6 * psutil.virtual_memory().total
    if args.no_e2e:
        fits = False
        e2e = dict(value=None, unit="routed tokens/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0, error="skipped (--no-e2e)")
    elif not fits:
        e2e = dict(value=None, unit="routed tokens/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0,
                   error="pinned host copies of the hidden states of all ranks do not fit host RAM")
    else:
        try:
            e2e = run_e2e(g, w, cfg, pc, st, hidden, off, cands, W, sb, slb, cur, dp, D, prev, out, delta, best, ws_r, ws_p, args, dev)
        except Exception as ex:  # report, never fake
            e2e = dict(value=None, unit="routed tokens/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0, error=str(ex)[:300])
    if dist and fits:
        e2e["ms_per_step"] = max_over_ranks(e2e["ms_per_step"], dev)
        e2e["value"] = replica_value(w.T, world, e2e["ms_per_step"])

    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            s, desc, threads, rates = oracle_step_time(w, *_sample(w))
            cpu = dict(value=w.T / s, unit="routed tokens/s", cores=threads, kind="oracle", sample=desc, **rates)
        line = dict(metric=METRIC, value=value, unit="routed tokens/s", n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                    ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16",
                    data="synthetic", config=_config(w, args), clocks=clocks, e2e=e2e, gpu_launches=int(launches),
                    roofline=roofline, cpu_baseline=cpu, token_layers_per_s=value * r.L, **extra)
        print(json.dumps(line))
    if dist:
        td.destroy_process_group()


def run_e2e(g, w, cfg, pc, st, hidden, off, cands, W, sb, slb, cur, dp, D, prev, out, delta, best, ws_r, ws_p, args, dev):
    r = w.router
    layer_bytes = w.T * r.H * 2
    hidden_host = torch.empty(hidden.shape, dtype=hidden.dtype, pin_memory=True)
    hidden_host.copy_(hidden)
    off_host = off.cpu().pin_memory()
    cands_host = torch.empty(cands.shape, dtype=cands.dtype, pin_memory=True)
    cands_host.copy_(cands)
    n_stage = 3
    stage = torch.empty(n_stage * layer_bytes, dtype=torch.uint8, device=dev)
    off_stage = torch.empty_like(off)
    cand_stage = torch.empty_like(cands)
    res_bytes = g.route_stats_result_bytes(cfg)
    result_host = torch.empty(res_bytes, dtype=torch.uint8, pin_memory=True)
    out_host = torch.empty(w.P, 5, dtype=torch.float32, pin_memory=True)
    argmin_host = torch.zeros(1, dtype=torch.int32, pin_memory=True)
    best_host = torch.zeros(r.L, dtype=torch.int32, pin_memory=True)
    torch.cuda.synchronize()

    ctx = g.HostCtx()

    def step():
        g.route_stats_host(ctx, cfg, st, T=w.T, hidden_host=hidden_host, src_offsets_host=off_host, hidden_stage=stage,
                           src_offsets_stage=off_stage, w_router=W, select_bias=sb, src_logit_bias=slb, cur_placement=cur,
                           dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, result_host=result_host, workspace=ws_r)
        A_live = st.A_step if w.mode == MODE_WINDOW else st.A_ema
        g.eval_placements_host(pc, cands_host, cand_stage, out, A_live, st.B, D, prev, out_host, argmin_host=argmin_host,
                               workspace=ws_p)
        g.eval_moves(pc, cur, prev, A_live, st.B, D, delta, best_per_layer=best, workspace=ws_p)
        best_host.copy_(best, non_blocking=True)
        torch.cuda.synchronize()

    step()                                                     # warm-up (stream / event creation, page touching)
    n = max(1, min(args.steps, 3))
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(n):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / n
    wall_ms = (time.perf_counter() - t0) * 1e3 / n
    h2d = hidden_host.numel() * 2 + off_host.numel() * 4 + cands_host.numel() * 2
    d2h = res_bytes + out_host.numel() * 4 + 4 + best_host.numel() * 4
    return dict(value=w.T / (ms * 1e-3), unit="routed tokens/s", h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                ms_per_step=ms, wall_ms_per_step=wall_ms, steps=n,
                note="gimbal_route_stats_host + gimbal_eval_placements_host + gimbal_eval_moves; pinned host buffers; "
                     "H2D of hidden overlaps the kernels layer by layer; bounded by the host link")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="v3", choices=["tiny", "v2lite", "qwen3", "v3", "decode"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--with-ids", action="store_true", help="also write top-k ids and weights (a2 outputs) inside the timed step")
    ap.add_argument("--layers", type=int, default=0, help="profiling only: run the first N MoE layers (named in config.workload)")
    args = ap.parse_args()
    w = get_workload(args.workload)
    if args.layers > 0:
        w = scaled(w, L=args.layers)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
