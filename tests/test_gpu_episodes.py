"""Multi-step episodes of the BASELINE.json configs through the real router-GEMM path (not synthetic logits):
  - DeepSeek-V2-Lite-shaped: EMA decay 0.9 over 32 steps, per-step lognormal source splits;
  - DeepSeek-V3-shaped: 24 steps, Zipf skew drifting every 8 steps, profiling windows of 8 steps;
  - decode-streaming: 256 tokens/step, EMA update every step, 200 consecutive steps replayed from ONE CUDA graph
    (the launch configuration of `bench.py --workload decode --episode`), a placement re-score every 100 steps.
Per step the fused kernel also writes its fp32 logits; the oracle checks them against its fp64 GEMM, gates on the same
fp32 logits (ids / counts bit-exact), and advances the window / EMA state, B and the per-source pressure in fp64.
Sizes are cut in L and T (and H for the 200-step run) so that the fp64 oracle GEMM finishes in seconds; T always spans
several 128-token tiles and a ragged tail.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_15177_b200 as g
from tests.test_gpu_parity import _check_objective, _logit_err, _oracle_kw
from tests.util import bf16_bits, to_np, ws_tensor
from workloads import gen, get_workload, scaled
from workloads.configs import MODE_EMA, MODE_WINDOW

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _oracle_step(r, hidden, W, slb, sb, off, logits_gpu):
    """oracle side of one step: logits (fp64) vs the GPU's, then gating + counts on the GPU's fp32 logits"""
    hb, wb, offn = bf16_bits(hidden), bf16_bits(W), to_np(off)
    Cs = np.empty((r.L, r.S, r.E), np.int64)
    worst = 0.0
    for l in range(r.L):
        l64, _ = oracle.router_logits(hb[l], wb[l], to_np(slb)[l], offn)
        worst = max(worst, _logit_err(to_np(logits_gpu[l]), l64))
        rid, _ = oracle.gate(to_np(logits_gpu[l]), r, None if sb is None else to_np(sb)[l], 1)
        Cs[l] = oracle.counts(rid, offn, r.S, r.E)
    return Cs, worst


def _run_episode(w, steps, window_len):
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    W = gen.w_router(w, DEV); sb = gen.select_bias(w, DEV); dp = gen.dp_of_rank(w, DEV)
    place = gen.prev_placement(w, np.random.default_rng(3).integers(1, 1000, (r.L, r.E)), DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    st = g.StatsState(cfg, w.mode, window_len=window_len, ema_decay=w.ema_decay)
    st_none = g.StatsState(cfg, w.mode, window_len=window_len, ema_decay=w.ema_decay)       # LOGITS_NONE twin (the bench path)
    logits = torch.empty(r.L, w.T, r.E, device=DEV)
    A_win = np.zeros((r.L, r.S, r.E), np.int64); A_pub = np.zeros_like(A_win); A_ema = np.zeros((r.L, r.S, r.E))
    published, biases = 0, []
    for step in range(steps):
        hidden = gen.hidden_all(w, step, DEV)
        slb = gen.src_logit_bias(w, step, DEV)
        off = gen.src_offsets(w, step, w.T, DEV)
        biases.append(to_np(slb))
        kw = dict(T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off, cur_placement=place,
                  dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws)
        g.route_stats(cfg, st, logits_mode=g.LOGITS_OUT, logits=logits, **kw)
        g.route_stats(cfg, st_none, **kw)
        torch.cuda.synchronize()
        Cs, worst = _oracle_step(r, hidden, W, slb, sb, off, logits)
        assert worst < 2e-4
        np.testing.assert_array_equal(to_np(st.A_step), Cs)
        assert torch.equal(st_none.A_step, st.A_step)
        if w.mode == MODE_WINDOW:
            live = A_win + Cs
            pub = oracle.update_window(A_win, Cs, A_pub, step, window_len)
            published += pub
            np.testing.assert_array_equal(to_np(st.A_win), A_win)
            np.testing.assert_array_equal(to_np(st.A_pub), A_pub)
            d = oracle.derived(live.astype(np.float64), to_np(place), to_np(dp), w.G, w.slots_per_rank)
            np.testing.assert_array_equal(to_np(st.B), d["B"].astype(np.int64))
            if pub:
                np.testing.assert_array_equal(to_np(st.B_pub), d["B"].astype(np.int64))
            assert torch.equal(st_none.A_win, st.A_win) and torch.equal(st_none.A_pub, st.A_pub)
        else:
            oracle.update_ema(A_ema, Cs, w.ema_decay)
            np.testing.assert_allclose(to_np(st.A_ema), A_ema, rtol=1e-5, atol=1e-30)
            d = oracle.derived(A_ema, to_np(place), to_np(dp), w.G, w.slots_per_rank)
            np.testing.assert_allclose(to_np(st.B), d["B"], rtol=1e-5)
            assert torch.equal(st_none.A_ema, st.A_ema)
        np.testing.assert_allclose(to_np(st.pressure_raw), d["pressure_raw"], rtol=1e-5)
        np.testing.assert_allclose(to_np(st.pressure_rel), d["pressure_rel"], rtol=1e-5)
        assert int(st.step_counter.item()) == step + 1 and int(st.status.item()) == 0
    return st, published, biases, place


def test_v2lite_episode_ema_over_32_steps():
    """BASELINE.json config 2: "EMA decay 0.9 over 32 steps", token counts per source from lognormal prompt lengths"""
    w = scaled(get_workload("v2lite"), L=2, T=700)
    assert w.mode == MODE_EMA and w.ema_decay == 0.9 and w.steps == 32
    st, _, _, _ = _run_episode(w, w.steps, window_len=1)
    # the un-normalised EMA of a stationary stream approaches C / (1 - d): after 32 steps the total is within 4 % of it
    total = float(st.A_ema.sum().item())
    assert abs(total / (w.router.L * w.T * w.router.k / (1 - 0.9)) - 1.0) < 0.04


def test_v3_episode_windows_and_drift_over_24_steps():
    """BASELINE.json config 4: "Zipf(1.3) skew drifting every 8 steps" over the proposed 24 steps, windows of 8 steps"""
    w = scaled(get_workload("v3"), L=2, T=300)
    assert w.mode == MODE_WINDOW and w.drift_every == 8 and w.steps == 24
    st, published, biases, _ = _run_episode(w, w.steps, window_len=8)
    assert published == 3
    # the skew really drifts at steps 8 and 16 and nowhere else
    changed = [not np.array_equal(biases[s], biases[s - 1]) for s in range(1, w.steps)]
    assert [s + 1 for s, c in enumerate(changed) if c] == [8, 16]
    assert int(st.A_win.abs().sum().item()) == 0                       # the last window was published and reset


def test_decode_episode_200_steps_from_one_cuda_graph():
    """BASELINE.json config 5 at reduced L / H: 256 tokens/step, EMA update every step, consecutive steps captured in ONE
    CUDA graph (10 steps reading a ring of 10 hidden-state buffers, the 100th step of every 100 also re-scores the
    candidates) and replayed 20 times = 200 steps; the oracle walks the same 200 steps."""
    w = scaled(get_workload("decode"), L=2, H=1024, P=96)
    r = w.router
    assert w.T == 256 and w.mode == MODE_EMA and w.rescore_every == 100
    cfg = g.RouterCfg.from_workload(r)
    ring, replays = 10, 20
    W = gen.w_router(w, DEV); sb = gen.select_bias(w, DEV); dp = gen.dp_of_rank(w, DEV)
    slb = gen.src_logit_bias(w, 0, DEV); off = gen.src_offsets(w, 0, w.T, DEV)
    place = gen.prev_placement(w, np.random.default_rng(4).integers(1, 1000, (r.L, r.E)), DEV)
    hidden = torch.stack([gen.hidden_all(w, s, DEV) for s in range(ring)])               # [ring, L, T, H]
    logits = torch.empty(ring, r.L, w.T, r.E, device=DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    pc = g.PlacementCfg(L=r.L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S, counts_dtype=g.COUNTS_F32)
    cands = gen.candidates(w, place, w.P, DEV)
    D = gen.comm_cost_D(w, "binary", DEV)
    wsp = ws_tensor(g.eval_placements_workspace_bytes(pc, w.P))
    out = torch.zeros(w.P, 5, device=DEV); argmin = torch.zeros(1, dtype=torch.int32, device=DEV)
    snap_A = torch.zeros(r.L, r.S, r.E, device=DEV); snap_B = torch.zeros(r.L, r.E, device=DEV)
    st = g.StatsState(cfg, MODE_EMA, ema_decay=w.ema_decay)
    # the bench's launch configuration of this regime: counts only (two epilogue warps per quadrant), counts stored through
    # distributed shared memory, programmatic dependent launches captured into the graph -- stepped beside the logits-out state
    st_b = g.StatsState(cfg, MODE_EMA, ema_decay=w.ema_decay)
    ws_b = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    g.set_option(g.OPT_PDL, 2)          # every input below is staged before the first launch (the promise GIMBAL_OPT_PDL = 2 asks for)
    g.kernel_timing(False)

    def ten_steps(stream, rescore):
        for i in range(ring):
            g.route_stats(cfg, st, T=w.T, hidden=hidden[i], w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                          logits_mode=g.LOGITS_OUT, logits=logits[i], cur_placement=place, dp_of_rank=dp, G=w.G,
                          slots_per_rank=w.slots_per_rank, workspace=ws, stream=stream)
            g.route_stats(cfg, st_b, T=w.T, hidden=hidden[i], w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                          cur_placement=place, dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws_b, stream=stream)
        if rescore:
            g.eval_placements(pc, cands, st.A_ema, st.B, D, place, out, argmin=argmin, workspace=wsp, stream=stream)
            with torch.cuda.stream(stream):
                snap_A.copy_(st.A_ema); snap_B.copy_(st.B)                                # the profile the re-score saw

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    ten_steps(side, True)                                                                 # warm-up outside the capture
    side.synchronize()
    graphs = {}
    for rescore in (False, True):
        graphs[rescore] = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graphs[rescore], stream=side):
            ten_steps(side, rescore)
    for t in (st.A_ema, st.B, st.A_step, st.step_counter, st.status, st_b.A_ema, st_b.B, st_b.A_step, st_b.step_counter, st_b.status):
        t.zero_()
    torch.cuda.synchronize()
    # per-step counts of the ring, once (the ring repeats every 10 steps)
    Cs = []
    A_ema = np.zeros((r.L, r.S, r.E))
    rescored = 0
    for rep in range(replays):
        rescore = ((rep + 1) * ring) % w.rescore_every == 0
        graphs[rescore].replay()
        torch.cuda.synchronize()
        if rep == 0:
            for i in range(ring):
                c, worst = _oracle_step(r, hidden[i], W, slb, sb, off, logits[i])
                assert worst < 2e-4
                Cs.append(c)
        for i in range(ring):
            oracle.update_ema(A_ema, Cs[i], w.ema_decay)
        np.testing.assert_allclose(to_np(st.A_ema), A_ema, rtol=1e-5, atol=1e-30)
        assert int(st.step_counter.item()) == (rep + 1) * ring
        assert torch.equal(st_b.A_ema, st.A_ema) and torch.equal(st_b.A_step, st.A_step) and torch.equal(st_b.B, st.B)
        assert torch.equal(st_b.pressure_rel, st.pressure_rel) and int(st_b.step_counter.item()) == (rep + 1) * ring
        if rescore:
            rescored += 1
            np.testing.assert_allclose(to_np(snap_A), A_ema, rtol=1e-5, atol=1e-30)
            ref = oracle.objective_batch(to_np(cands), to_np(place), to_np(snap_A), to_np(snap_B), to_np(D), None, 1.0, **_oracle_kw(pc))
            _check_objective(to_np(out).astype(np.float64), ref)
            assert int(argmin.item()) == int(np.argmin(to_np(out)[:, 0]))
    assert rescored == 2 and int(st.status.item()) == 0
    d = oracle.derived(A_ema, to_np(place), to_np(dp), w.G, w.slots_per_rank)
    np.testing.assert_allclose(to_np(st.B), d["B"], rtol=1e-5)
    np.testing.assert_allclose(to_np(st.pressure_rel), d["pressure_rel"], rtol=1e-5)


@pytest.mark.parametrize("name,T,L,window_len", [("v3", 256, 3, 2), ("v3", 100, 2, 3), ("decode", 256, 4, 1), ("qwen3", 200, 3, 2),
                                                   ("qwen3", 128, 2, 2), ("v2lite", 77, 3, 2), ("tiny", 200, 1, 1), ("tiny", 64, 1, 2)])
def test_small_batch_regime_fused_update_matches_the_separate_kernels(name, T, L, window_len):
    """One tile per layer (T <= 256, every layer with a CTA pair of its own): the router kernel stores the counts (no zeroing of
    A_step) and, in a whole-step call, runs the window / EMA update of its layer in its tail (GIMBAL_OPT_FUSE_UPDATE).  Six steps
    beside a state driven with the option off and programmatic launches off (memset-free store path + separate
    stats_update_kernel) and a third one fed layer by layer (sliced calls: separate update kernel): every state array bit for bit,
    incl. the publish / reset steps of the window mode; the counts against the oracle on the GPU's logits.  T <= 128 takes the
    cta_group::1 kernel."""
    w = scaled(get_workload(name), L=L, T=T)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    W = gen.w_router(w, DEV); sb = gen.select_bias(w, DEV); dp = gen.dp_of_rank(w, DEV)
    place = gen.prev_placement(w, np.random.default_rng(5).integers(1, 1000, (r.L, r.E)), DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    states = [g.StatsState(cfg, w.mode, window_len=window_len, ema_decay=w.ema_decay) for _ in range(3)]
    logits = torch.empty(r.L, w.T, r.E, device=DEV)
    st_l = g.StatsState(cfg, w.mode, window_len=window_len, ema_decay=w.ema_decay)
    for step in range(6):
        hidden = gen.hidden_all(w, step, DEV); slb = gen.src_logit_bias(w, step, DEV); off = gen.src_offsets(w, step, w.T, DEV)
        kw = dict(T=w.T, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off, cur_placement=place, dp_of_rank=dp, G=w.G,
                  slots_per_rank=w.slots_per_rank, workspace=ws)
        g.set_option(g.OPT_FUSE_UPDATE, 1); g.set_option(g.OPT_PDL, 1)
        g.route_stats(cfg, states[0], hidden=hidden, **kw)
        g.route_stats(cfg, st_l, hidden=hidden, logits_mode=g.LOGITS_OUT, logits=logits, **kw)
        g.set_option(g.OPT_FUSE_UPDATE, 0); g.set_option(g.OPT_PDL, 0)
        g.route_stats(cfg, states[1], hidden=hidden, **kw)
        g.set_option(g.OPT_FUSE_UPDATE, 1); g.set_option(g.OPT_PDL, 1)
        for l in range(r.L):
            g.route_stats(cfg, states[2], hidden=hidden[l:l + 1], layer0=l, n_layers=1, **kw)
        torch.cuda.synchronize()
        offn = to_np(off)
        for l in range(r.L):
            rid, _ = oracle.gate(to_np(logits[l]), r, None if sb is None else to_np(sb)[l], 1)
            np.testing.assert_array_equal(to_np(states[0].A_step[l]), oracle.counts(rid, offn, r.S, r.E))
        for other in states[1:] + [st_l]:
            for f in ("A_step", "A_win", "A_pub", "B_pub", "A_ema", "B", "pressure_raw", "pressure_rel", "step_counter", "status"):
                assert torch.equal(getattr(other, f), getattr(states[0], f)), (step, f)
        assert int(states[0].step_counter.item()) == step + 1 and int(states[0].status.item()) == 0
        assert int(states[0]._step_words[1].item()) == 0                      # the library's layer counter is 0 between calls
