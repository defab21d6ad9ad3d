"""Parity at BASELINE.json's FULL size, in the launch configuration bench.py times (DeepSeek-V3-shaped:
58 layers, hidden 7168, 256 experts, 65536 tokens/step, 288 slots on 32 ranks, 4096 candidates, the whole
move neighbourhood).  The oracle cannot redo 14 TFLOP of fp64 GEMM, so:
  - properties that hold at any size are checked on ALL outputs of the bench-configuration call;
  - a second call that also writes logits and ids must reproduce the same counts bit for bit, and on SAMPLED
    layers / rows the oracle recomputes the logits (fp64), the gating (bit-exact on the GPU's logits) and the
    counts (bit-exact, full layer);
  - sampled candidates and sampled moves of the full-size placement calls are recomputed by the oracle.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_15177_b200 as g
from tests.test_gpu_parity import _check_deltas, _check_objective, _logit_err, _oracle_kw
from tests.util import bf16_bits, to_np, ws_tensor
from workloads import gen, get_workload
from workloads.configs import MODE_WINDOW

pytestmark = pytest.mark.gpu
DEV = "cuda"


def test_v3_full_size_bench_configuration():
    if torch.cuda.get_device_properties(0).total_memory < 100e9:
        pytest.skip("needs the 54.5 GB of hidden states of the V3 config resident")
    w = get_workload("v3")
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    hidden = gen.hidden_all(w, 0, DEV)
    W = gen.w_router(w, DEV)
    slb = gen.src_logit_bias(w, 0, DEV)
    sb = gen.select_bias(w, DEV)
    off = gen.src_offsets(w, 0, w.T, DEV)
    dp = gen.dp_of_rank(w, DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    st = g.StatsState(cfg, MODE_WINDOW, window_len=8)
    prev0 = gen.prev_placement(w, np.ones((r.L, r.E)), DEV)
    # ---- the bench call: fused, nothing but the counts leaves the chip
    g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                  cur_placement=prev0, dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws)
    torch.cuda.synchronize()
    A = to_np(st.A_step).astype(np.int64)
    offn = to_np(off)
    assert int(st.status.item()) == 0 and int(st.step_counter.item()) == 1
    assert (A >= 0).all()
    np.testing.assert_array_equal(A.sum(2), np.broadcast_to(np.diff(offn) * r.k, (r.L, r.S)))      # row sums = tokens x k
    assert A.sum() == r.L * w.T * r.k
    np.testing.assert_array_equal(to_np(st.B), A.sum(1))                                             # B = sum_s A
    np.testing.assert_array_equal(to_np(st.A_win), A)
    d = oracle.derived(A.astype(np.float64), to_np(prev0), to_np(dp), w.G, w.slots_per_rank)
    np.testing.assert_allclose(to_np(st.pressure_raw), d["pressure_raw"], rtol=1e-5)
    np.testing.assert_allclose(to_np(st.pressure_rel), d["pressure_rel"], rtol=1e-5)
    np.testing.assert_allclose(to_np(st.pressure_raw).sum(), A.sum(), rtol=1e-5)                     # loads sum to routed tokens

    # ---- two epilogue warps per quadrant (GIMBAL_OPT_EPI_PARTS = 2, normally the small-batch kernel) over all 14,848 tiles
    g.set_option(g.OPT_EPI_PARTS, 2)
    st_p = g.StatsState(cfg, MODE_WINDOW, window_len=8)
    g.route_stats(cfg, st_p, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off, workspace=ws)
    g.set_option(g.OPT_EPI_PARTS, 0)
    assert torch.equal(st_p.A_step, st.A_step)

    # ---- sampled layers: logits + ids written by a layer-sliced call must give the same counts; oracle on samples
    rng = np.random.default_rng(0)
    for l in sorted(rng.choice(r.L, 3, replace=False).tolist()):
        st1 = g.StatsState(cfg, MODE_WINDOW, window_len=8)
        logits = torch.empty(1, w.T, r.E, device=DEV)
        ids = torch.empty(1, w.T, r.k, dtype=torch.int32, device=DEV)
        g.route_stats(cfg, st1, T=w.T, hidden=hidden[l:l + 1], w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                      layer0=l, n_layers=1, logits_mode=g.LOGITS_OUT, logits=logits, topk_ids=ids, workspace=ws)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(to_np(st1.A_step[l]), A[l])                                   # same counts, bit for bit
        gl, gi = to_np(logits[0]), to_np(ids[0])
        rows = np.unique(np.concatenate([rng.integers(0, w.T, 192), [0, 127, 128, w.T - 1], offn[1:-1], offn[1:-1] - 1]))
        rows = rows[(rows >= 0) & (rows < w.T)]
        hb = bf16_bits(hidden[l][torch.from_numpy(rows).to(DEV)])
        src_rows = np.searchsorted(offn, rows, side="right") - 1
        # fp64 logits of the sampled rows: bias of each row's own source
        for s in np.unique(src_rows):
            m = src_rows == s
            l64, _ = oracle.router_logits(hb[m], bf16_bits(W[l]), to_np(slb)[l][s:s + 1], np.array([0, int(m.sum())], np.int32))
            assert _logit_err(gl[rows[m]], l64) < 2e-4
        rid, _ = oracle.gate(gl, r, to_np(sb)[l], 1)                                                # whole layer, on the GPU's logits
        np.testing.assert_array_equal(gi, rid)
        np.testing.assert_array_equal(oracle.counts(rid, offn, r.S, r.E), A[l])

    # ---- placement side at full size on the profile just collected
    pc = g.PlacementCfg(L=r.L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S)
    Dm = gen.comm_cost_D(w, "binary", DEV)
    prev = gen.prev_placement(w, to_np(st.B), DEV)
    cands = gen.candidates(w, prev, w.P, DEV)
    out = torch.empty(w.P, 5, device=DEV)
    argmin = torch.zeros(1, dtype=torch.int32, device=DEV)
    wsp = ws_tensor(g.eval_placements_workspace_bytes(pc, w.P))
    g.eval_placements(pc, cands, st.A_step, st.B, Dm, prev, out, argmin=argmin, workspace=wsp)
    o = to_np(out).astype(np.float64)
    assert not np.isnan(o).any() and o[0, 3] == 0.0                                                 # all valid; C_mig(x0) = 0
    assert int(argmin.item()) == int(np.argmin(to_np(out)[:, 0]))
    pick = np.unique(np.concatenate([[0, 1, w.P // 2, w.P - 1], rng.integers(0, w.P, 28)]))
    ref = oracle.objective_batch(to_np(cands)[pick], to_np(prev), A, A.sum(1), to_np(Dm), None, 1.0, **_oracle_kw(pc))
    _check_objective(o[pick], ref)
    assert np.allclose(o[:, 2] + 0.0, o[:, 2]) and (o[:, 2] <= A.sum() * (1 + 1e-6)).all()          # binary D: C_comm <= all routed tokens

    cur = cands[2].contiguous()
    n = r.L * w.NS * (w.NS - 1) // 2
    delta = torch.empty(n, 5, device=DEV)
    best = torch.empty(r.L, dtype=torch.int32, device=DEV)
    g.eval_moves(pc, cur, prev, st.A_step, st.B, Dm, delta, best_per_layer=best, workspace=wsp)
    dl = to_np(delta)
    allmv = oracle.all_pair_moves(r.L, w.NS)
    pickm = np.unique(np.concatenate([np.arange(200), np.arange(n - 200, n), rng.integers(0, n, 1600)]))
    refm = oracle.move_deltas(to_np(cur), to_np(prev), allmv[pickm], A, A.sum(1), to_np(Dm), None, 1.0, **_oracle_kw(pc))
    _check_deltas(pc, dl[pickm].astype(np.float64), refm, allmv[pickm], to_np(cur), A, A.sum(1), to_np(Dm), None, 1.0)
    per = n // r.L
    for l in range(r.L):
        assert int(best[l].item()) == l * per + int(np.nanargmin(dl[l * per:(l + 1) * per, 0]))


@pytest.mark.parametrize("name", ["tiny", "v2lite", "qwen3", "decode"])
def test_other_configs_full_size_bench_configuration(name):
    """BASELINE.json configs 1, 2, 3 and 5 at their stated sizes (every layer, all tokens of a step, all P candidates, the
    whole move neighbourhood), in the call bench.py makes for `--workload <name>`: invariants on ALL outputs; on sampled
    layers the oracle redoes the gating and the counts of the WHOLE layer on the GPU's own logits (bit-exact) and the fp64
    logits of sampled rows; sampled candidates and moves of the full-size placement calls."""
    w = get_workload(name)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    hidden = gen.hidden_all(w, 0, DEV)
    W = gen.w_router(w, DEV)
    slb = gen.src_logit_bias(w, 0, DEV)
    sb = gen.select_bias(w, DEV)
    off = gen.src_offsets(w, 0, w.T, DEV)
    dp = gen.dp_of_rank(w, DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    mk = lambda: g.StatsState(cfg, w.mode, window_len=w.window_len, ema_decay=w.ema_decay)
    st = mk()
    prev0 = gen.prev_placement(w, np.ones((r.L, r.E)), DEV)
    g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                  cur_placement=prev0, dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws)
    torch.cuda.synchronize()
    A = to_np(st.A_step).astype(np.int64)
    offn = to_np(off)
    assert int(st.status.item()) == 0 and int(st.step_counter.item()) == 1
    assert (A >= 0).all()
    np.testing.assert_array_equal(A.sum(2), np.broadcast_to(np.diff(offn) * r.k, (r.L, r.S)))      # row sums = tokens x k
    assert A.sum() == r.L * w.T * r.k
    if w.mode == MODE_WINDOW:
        np.testing.assert_array_equal(to_np(st.B), A.sum(1))                                         # B = sum_s A
        if w.window_len == 1:                                                                        # published and reset at once
            np.testing.assert_array_equal(to_np(st.A_pub), A)
            assert not to_np(st.A_win).any()
        else:
            np.testing.assert_array_equal(to_np(st.A_win), A)
    else:                                                                                            # first EMA step from zero: A = C
        np.testing.assert_array_equal(to_np(st.A_ema), A.astype(np.float32))
        np.testing.assert_allclose(to_np(st.B), A.sum(1), rtol=1e-6)
    d = oracle.derived(A.astype(np.float64), to_np(prev0), to_np(dp), w.G, w.slots_per_rank)
    np.testing.assert_allclose(to_np(st.pressure_raw), d["pressure_raw"], rtol=1e-5)
    np.testing.assert_allclose(to_np(st.pressure_rel), d["pressure_rel"], rtol=1e-5)
    np.testing.assert_allclose(to_np(st.pressure_raw).sum(), A.sum(), rtol=1e-5)                     # loads sum to routed tokens

    rng = np.random.default_rng(1)
    sbn = None if sb is None else to_np(sb)
    for l in sorted(rng.choice(r.L, min(r.L, 3), replace=False).tolist()):
        st1 = mk()
        logits = torch.empty(1, w.T, r.E, device=DEV)
        ids = torch.empty(1, w.T, r.k, dtype=torch.int32, device=DEV)
        g.route_stats(cfg, st1, T=w.T, hidden=hidden[l:l + 1], w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                      layer0=l, n_layers=1, logits_mode=g.LOGITS_OUT, logits=logits, topk_ids=ids, workspace=ws)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(to_np(st1.A_step[l]), A[l])                                   # same counts, bit for bit
        gl, gi = to_np(logits[0]), to_np(ids[0])
        rows = np.unique(np.concatenate([rng.integers(0, w.T, 192), [0, 127, 128, w.T - 1], offn[1:-1], offn[1:-1] - 1]))
        rows = rows[(rows >= 0) & (rows < w.T)]
        hb = bf16_bits(hidden[l][torch.from_numpy(rows).to(DEV)])
        src_rows = np.searchsorted(offn, rows, side="right") - 1
        for s in np.unique(src_rows):
            m = src_rows == s
            l64, _ = oracle.router_logits(hb[m], bf16_bits(W[l]), to_np(slb)[l][s:s + 1], np.array([0, int(m.sum())], np.int32))
            assert _logit_err(gl[rows[m]], l64) < 2e-4
        rid, _ = oracle.gate(gl, r, None if sbn is None else sbn[l], 1)                             # whole layer, on the GPU's logits
        np.testing.assert_array_equal(gi, rid)
        np.testing.assert_array_equal(oracle.counts(rid, offn, r.S, r.E), A[l])

    # ---- placement side at full size on the profile just collected
    pc = g.PlacementCfg(L=r.L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S)
    Dm = gen.comm_cost_D(w, "binary", DEV)
    Bn = A.sum(1)
    prev = gen.prev_placement(w, Bn, DEV)
    cands = gen.candidates(w, prev, w.P, DEV)
    out = torch.empty(w.P, 5, device=DEV)
    argmin = torch.zeros(1, dtype=torch.int32, device=DEV)
    wsp = ws_tensor(g.eval_placements_workspace_bytes(pc, w.P))
    Bt = torch.from_numpy(Bn.astype(np.int32)).to(DEV)
    g.eval_placements(pc, cands, st.A_step, Bt, Dm, prev, out, argmin=argmin, workspace=wsp)
    o = to_np(out).astype(np.float64)
    assert not np.isnan(o).any() and o[0, 3] == 0.0                                                 # all valid; C_mig(x0) = 0
    assert int(argmin.item()) == int(np.argmin(to_np(out)[:, 0]))
    pick = np.unique(np.concatenate([[0, 1, w.P // 2, w.P - 1], rng.integers(0, w.P, 28)]))
    ref = oracle.objective_batch(to_np(cands)[pick], to_np(prev), A, Bn, to_np(Dm), None, 1.0, **_oracle_kw(pc))
    _check_objective(o[pick], ref)
    assert (o[:, 2] <= A.sum() * (1 + 1e-6)).all()                                                  # binary D: C_comm <= all routed tokens

    cur = cands[2].contiguous()
    n = r.L * w.NS * (w.NS - 1) // 2
    delta = torch.empty(n, 5, device=DEV)
    best = torch.empty(r.L, dtype=torch.int32, device=DEV)
    g.eval_moves(pc, cur, prev, st.A_step, Bt, Dm, delta, best_per_layer=best, workspace=wsp)
    dl = to_np(delta)
    allmv = oracle.all_pair_moves(r.L, w.NS)
    pickm = np.unique(np.concatenate([np.arange(min(n, 200)), np.arange(max(0, n - 200), n), rng.integers(0, n, 1600)]))
    refm = oracle.move_deltas(to_np(cur), to_np(prev), allmv[pickm], A, Bn, to_np(Dm), None, 1.0, **_oracle_kw(pc))
    _check_deltas(pc, dl[pickm].astype(np.float64), refm, allmv[pickm], to_np(cur), A, Bn, to_np(Dm), None, 1.0)
    per = n // r.L
    for l in range(r.L):
        assert int(best[l].item()) == l * per + int(np.nanargmin(dl[l * per:(l + 1) * per, 0]))
