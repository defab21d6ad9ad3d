"""GPU parity tests: the CUDA path (through the C-ABI binding) against the CPU oracle,
element by element on the same seeded inputs.

Bars (BASELINE.json north_star): integer / index work bit-exact; router logits within 1e-2
relative (bf16 inputs, fp32 accumulation); fp32 objectives within 1e-5 relative to the oracle's
value (move DELTAS, which are differences by definition, relative to the magnitude of the terms that
were added, R13).

Order matters on a fresh box: placement and gating kernels first, the tcgen05 GEMM last.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_15177_b200 as g
from tests.util import bf16_bits, to_np, ws_tensor
from workloads import gen, get_workload, scaled
from workloads.configs import MODE_EMA, MODE_WINDOW, SIGMOID

pytestmark = pytest.mark.gpu
DEV = "cuda"

SHAPES = {                      # name -> (L, T, P) scaled so the oracle finishes in seconds
    "tiny": (1, 1000, 64),
    "v2lite": (3, 1500, 96),
    "qwen3": (2, 1300, 64),
    "v3": (2, 1100, 48),
    "decode": (2, 256, 64),
}


def _wl(name):
    L, T, P = SHAPES[name]
    return scaled(get_workload(name), L=L, T=T, P=P)


# ------------------------------------------------------------------------------------------
# placement side (a6, a7)
# ------------------------------------------------------------------------------------------
def _placement_instance(name, seed=0, counts="i32", table_M=False, seeded_D=False):
    w = _wl(name)
    r = w.router
    rng = np.random.default_rng(100 + seed)
    # counts shaped like a skewed routing profile; B lives on another scale than A
    pop = rng.zipf(1.3, size=(r.L, r.E)).clip(1, 500).astype(np.float64)
    A = (rng.random((r.L, r.S, r.E)) * pop[:, None, :] * 40).astype(np.int64)
    B = A.sum(1) * rng.integers(50, 150, (r.L, r.E))
    if counts == "f32":
        A_t = torch.from_numpy((A * 0.37).astype(np.float32)).to(DEV)
        B_t = torch.from_numpy((B * 0.37).astype(np.float32)).to(DEV)
    else:
        A_t = torch.from_numpy(A.astype(np.int32)).to(DEV)
        B_t = torch.from_numpy(B.astype(np.int32)).to(DEV)
    D = gen.comm_cost_D(w, "seeded" if seeded_D else "binary", DEV)
    M = gen.mig_cost_M(w, DEV) if table_M else None
    prev = gen.prev_placement(w, to_np(B_t), DEV)
    cfg = g.PlacementCfg(L=r.L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S,
                         counts_dtype=g.COUNTS_F32 if counts == "f32" else g.COUNTS_I32)
    return w, cfg, A_t, B_t, D, M, prev


def _oracle_kw(cfg):
    return dict(G=cfg.G, sp=cfg.slots_per_rank, weights=(cfg.alpha, cfg.beta, cfg.gamma))


def _check_objective(out, ref, tol=1e-5):
    """out, ref [P,5] = {J, C_load, C_comm, C_mig, maxload}: NaN exactly where the oracle says, every column within
    `tol` of the oracle's value (BASELINE.json: "fp32 objectives within 1e-5 relative").  C_load is a sum of squares of
    differences of rank loads: where the loads are balanced to better than fp32 resolution its scale is floored at
    1e-6 * maxload^2 (R11)."""
    assert np.array_equal(np.isnan(out), np.isnan(ref))
    ok = ~np.isnan(ref[:, 0])
    scale = np.abs(ref[ok])
    err = np.abs(out[ok] - ref[ok])
    assert np.all(err[:, [0, 2, 3, 4]] <= tol * scale[:, [0, 2, 3, 4]]), (err / (scale + 1e-300)).max(0)
    load_scale = np.maximum(np.abs(ref[ok, 1]), 1e-6 * np.abs(ref[ok, 4]) ** 2)
    assert np.all(np.abs(out[ok, 1] - ref[ok, 1]) <= tol * load_scale)


PLACEMENT_CASES = [
    ("tiny", "i32", False, False), ("v2lite", "f32", True, True), ("qwen3", "i32", False, True),
    ("v3", "i32", False, False), ("v3", "f32", True, True), ("decode", "f32", False, False), ("decode", "i32", True, True),
]


@pytest.mark.parametrize("name,counts,table_M,seeded_D", PLACEMENT_CASES)
@pytest.mark.parametrize("kernel", ["fast", "generic", "check_scores_all", "trusted"])
def test_eval_placements_parity(name, counts, table_M, seeded_D, kernel):
    """a6 against the oracle; the specialised and the shape-generic scoring kernel, the validation kernel's own
    scoring (candidate's r from its bit matrix), and the GIMBAL_PLACE_TRUSTED call that skips validation."""
    g.set_option(g.OPT_SCORE_GENERIC, int(kernel == "generic"))
    g.set_option(g.OPT_CHECK_SCORES_ALL, int(kernel == "check_scores_all"))
    w, cfg, A, B, D, M, prev = _placement_instance(name, 0, counts, table_M, seeded_D)
    if kernel == "trusted":
        cfg.flags = g.PLACE_TRUSTED
    cands = gen.candidates(w, prev, w.P, DEV)
    out = torch.full((w.P, 5), -1.0, device=DEV)
    argmin = torch.full((1,), -7, dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.eval_placements_workspace_bytes(cfg, w.P))
    g.eval_placements(cfg, cands, A, B, D, prev, out, M=M, M_scalar=1.25, argmin=argmin, workspace=ws)
    torch.cuda.synchronize()
    ref = oracle.objective_batch(to_np(cands), to_np(prev), to_np(A), to_np(B), to_np(D), to_np(M), 1.25, **_oracle_kw(cfg))
    o = to_np(out).astype(np.float64)
    _check_objective(o, ref)
    assert o[0, 3] == 0.0                                   # candidate 0 is x0: migration cost is 0 for an unchanged placement
    # argmin: lowest index among the minimisers of the GPU's own J; its oracle J is the oracle minimum (to tolerance)
    am = int(argmin.item())
    assert am == int(np.nanargmin(to_np(out)[:, 0]))
    assert ref[am, 0] <= np.nanmin(ref[:, 0]) * (1 + 2e-5)


@pytest.mark.parametrize("name,counts,table_M,seeded_D", [("v3", "i32", False, False), ("v3", "f32", True, True), ("decode", "i32", True, True),
                                                            ("qwen3", "i32", False, True)])
def test_eval_placements_candidates_with_their_own_replica_sets(name, counts, table_M, seeded_D):
    """DESIGN.md R12 / SURVEY 8c #12: r[l,e] is the candidate's.  Every (candidate, layer) re-draws its redundant copies
    (an expert may get 3+ ranks); the oracle scores them and so must the GPU.  Without redundant slots (decode, qwen3)
    the same generator gives plain permutations."""
    w, cfg, A, B, D, M, prev = _placement_instance(name, 7, counts, table_M, seeded_D)
    cands = gen.candidates_redrawn(w, prev, w.P, DEV)
    if w.NS > cfg.E:
        c0, p0 = to_np(cands[1, 0]), to_np(prev[0])
        assert sorted(c0.tolist()) != sorted(p0.tolist()) and np.bincount(c0, minlength=cfg.E).max() >= 2
    out = torch.empty(w.P, 5, device=DEV)
    argmin = torch.zeros(1, dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.eval_placements_workspace_bytes(cfg, w.P))
    g.eval_placements(cfg, cands, A, B, D, prev, out, M=M, M_scalar=0.5, argmin=argmin, workspace=ws)
    ref = oracle.objective_batch(to_np(cands), to_np(prev), to_np(A), to_np(B), to_np(D), to_np(M), 0.5, **_oracle_kw(cfg))
    o = to_np(out).astype(np.float64)
    assert not np.isnan(ref).any()
    _check_objective(o, ref)
    assert o[0, 3] == 0.0 and int(argmin.item()) == int(np.argmin(to_np(out)[:, 0]))


def test_eval_placements_invalid_candidates_and_edges():
    w, cfg, A, B, D, M, prev = _placement_instance("v3", 1)
    P = 40
    cands = gen.candidates(w, prev, P, DEV).clone()
    NS, sp = w.NS, w.slots_per_rank
    cands[3, 0, 5] = 300                                   # id out of range
    cands[4, 1, 7] = -2
    c5 = cands[5, 0].clone(); c5[0] = c5[1]; cands[5, 0] = c5            # expert twice on a rank (and one missing)
    # a co-located duplicate that keeps the multiset: exchange so that both copies of a replicated expert share a rank
    row = to_np(cands[6, 1]).copy()
    vals, cnt = np.unique(row, return_counts=True)
    e = vals[cnt == 2][0]
    j0, j1 = np.nonzero(row == e)[0]
    tgt = (j0 // sp) * sp + ((j0 % sp) + 1) % sp           # another slot on j0's rank
    row[j1], row[tgt] = row[tgt], row[j1]
    cands[6, 1] = torch.from_numpy(row).to(DEV)
    # an expert hosted nowhere, no rank holding anything twice: a singly-hosted expert's slot takes a copy of an expert
    # that lives on other ranks
    row = to_np(cands[7, 0]).copy()
    vals, cnt = np.unique(row, return_counts=True)
    single = vals[cnt == 1][0]
    js = int(np.nonzero(row == single)[0][0])
    on_rank = set(row[(js // sp) * sp:(js // sp + 1) * sp].tolist())
    row[js] = next(int(v) for v in vals if int(v) not in on_rank)
    cands[7, 0] = torch.from_numpy(row).to(DEV)
    # valid, but another replica set than x0: one copy of a replicated expert becomes a second copy of a single one
    row = to_np(cands[8, 0]).copy()
    vals, cnt = np.unique(row, return_counts=True)
    dbl = vals[cnt == 2][0]
    jd = int(np.nonzero(row == dbl)[0][0])
    on_rank = set(row[(jd // sp) * sp:(jd // sp + 1) * sp].tolist())
    row[jd] = next(int(v) for v in vals[cnt == 1] if int(v) not in on_rank)
    cands[8, 0] = torch.from_numpy(row).to(DEV)
    out = torch.empty(P, 5, device=DEV)
    ws = ws_tensor(g.eval_placements_workspace_bytes(cfg, P))
    g.eval_placements(cfg, cands, A, B, D, prev, out, workspace=ws)
    ref = oracle.objective_batch(to_np(cands), to_np(prev), to_np(A), to_np(B), to_np(D), None, 1.0, **_oracle_kw(cfg))
    o = to_np(out).astype(np.float64)
    assert np.isnan(ref[[3, 4, 5, 6, 7]]).all() and not np.isnan(ref[8]).any()
    _check_objective(o, ref)                               # NaN exactly where the oracle says, values everywhere else
    # GIMBAL_PLACE_TRUSTED skips the validation: invalid rows get finite garbage, never a fault; valid rows are unchanged
    cfg_t = g.PlacementCfg(**{**cfg.__dict__, "flags": g.PLACE_TRUSTED})
    out_t = torch.empty(P, 5, device=DEV)
    g.eval_placements(cfg_t, cands, A, B, D, prev, out_t, workspace=ws)
    torch.cuda.synchronize()
    good = [p for p in range(P) if p not in (3, 4, 5, 6, 7, 8)]
    assert torch.equal(out_t[good], out[good])
    # P = 0 is a no-op; P = 1 works
    g.eval_placements(cfg, cands[:0], A, B, D, prev, out[:0], workspace=ws)
    g.eval_placements(cfg, cands[:1], A, B, D, prev, out[:1], workspace=ws)
    np.testing.assert_allclose(to_np(out[0]).astype(np.float64), ref[0], rtol=1e-5)
    # an invalid x0 poisons everything
    bad_prev = prev.clone(); bad_prev[0, 0] = bad_prev[0, 1]
    g.eval_placements(cfg, cands[:4], A, B, D, bad_prev, out[:4], workspace=ws)
    assert torch.isnan(out[:4]).all()


@pytest.mark.parametrize("name,counts,table_M,seeded_D", [c for c in PLACEMENT_CASES if c[0] != "v3"])
def test_eval_placements_expert_to_rank_u8_encoding(name, counts, table_M, seeded_D):
    """SURVEY 8b's second candidate encoding ([P,L,E] uint8, expert -> rank; configs without replicas): same values as
    the oracle on the equivalent slot -> expert rows, NaN for a rank out of range or over capacity."""
    w, cfg, A, B, D, M, prev = _placement_instance(name, 8, counts, table_M, seeded_D)
    cands = gen.candidates(w, prev, w.P, DEV)
    u8 = gen.to_expert_rank_u8(cands, w.slots_per_rank)
    bad = u8.clone()
    bad[3, 0, 5] = cfg.G                                                      # rank out of range
    e0 = int(to_np(prev)[0, 0])                                               # expert of slot 0 (rank 0) ...
    bad[4, 0, :] = u8[0, 0, :]; bad[4, 0, e0] = 1 if cfg.G > 1 else 0          # ... sent to rank 1: rank 1 over capacity
    cfg8 = g.PlacementCfg(**{**cfg.__dict__, "encoding": g.ENC_EXPERT_TO_RANK_U8})
    out = torch.empty(w.P, 5, device=DEV)
    argmin = torch.zeros(1, dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.eval_placements_workspace_bytes(cfg8, w.P))
    g.eval_placements(cfg8, bad, A, B, D, prev, out, M=M, M_scalar=1.25, argmin=argmin, workspace=ws)
    ref = oracle.objective_batch(to_np(cands), to_np(prev), to_np(A), to_np(B), to_np(D), to_np(M), 1.25, **_oracle_kw(cfg))
    ref[[3, 4]] = np.nan
    o = to_np(out).astype(np.float64)
    _check_objective(o, ref)
    assert o[0, 3] == 0.0 and int(argmin.item()) == int(np.nanargmin(to_np(out)[:, 0]))
    cfg8.flags = g.PLACE_TRUSTED
    out_t = torch.empty(w.P, 5, device=DEV)
    g.eval_placements(cfg8, u8, A, B, D, prev, out_t, M=M, M_scalar=1.25, workspace=ws)
    ref = oracle.objective_batch(to_np(cands), to_np(prev), to_np(A), to_np(B), to_np(D), to_np(M), 1.25, **_oracle_kw(cfg))
    _check_objective(to_np(out_t).astype(np.float64), ref)


def _delta_scales(cfg, moves, cur, A, B, D, M, M_scalar):
    """|terms| that a delta is made of (tolerance base, R13)."""
    L, E, G, sp = cfg.L, cfg.E, cfg.G, cfg.slots_per_rank
    A = A.astype(np.float64); B = B.astype(np.float64); D = D.astype(np.float64)
    r = np.stack([np.bincount(cur[l], minlength=E) for l in range(L)]).astype(np.float64)
    w = B / r
    Lg = np.stack([[w[l, cur[l, gidx * sp:(gidx + 1) * sp]].sum() for gidx in range(G)] for l in range(L)])
    c = np.einsum("lse,sg->leg", A, D) / r[:, :, None]
    sc = np.zeros((len(moves), 5))
    for i, (l, a, b) in enumerate(moves):
        e1, e2, g1, g2 = cur[l, a], cur[l, b], a // sp, b // sp
        dl = w[l, e2] - w[l, e1]
        sc[i, 1] = abs(2 * dl * (Lg[l, g1] - Lg[l, g2])) + 2 * dl * dl
        sc[i, 2] = c[l, e1, g1] + c[l, e1, g2] + c[l, e2, g1] + c[l, e2, g2]
        sc[i, 3] = 4 * (M_scalar if M is None else M[l].max())
        sc[i, 4] = Lg[l].max()
        sc[i, 0] = cfg.alpha * sc[i, 2] + cfg.beta * sc[i, 1] + cfg.gamma * sc[i, 3]
    return sc


def _check_deltas(cfg, d, ref, moves, cur, A, B, D, M, M_scalar, tol=1e-5):
    assert np.array_equal(np.isnan(d), np.isnan(ref))
    ok = ~np.isnan(ref[:, 0])
    sc = _delta_scales(cfg, moves[ok], cur, A, B, D, M, M_scalar)
    err = np.abs(d[ok] - ref[ok])
    assert np.all(err <= tol * sc + 1e-30), (err / (sc + 1e-30)).max(0)


@pytest.mark.parametrize("name,counts,table_M", [("tiny", "i32", False), ("v2lite", "f32", True), ("v3", "i32", False),
                                                   ("v3", "f32", True), ("decode", "i32", False)])
def test_eval_moves_parity(name, counts, table_M):
    w, cfg, A, B, D, M, prev = _placement_instance(name, 2, counts, table_M, True)
    cur = gen.candidates(w, prev, 4, DEV)[2].contiguous()          # a few transpositions away from x0
    kw = _oracle_kw(cfg)
    An, Bn, Dn, Mn, curn, prevn = to_np(A), to_np(B), to_np(D), to_np(M), to_np(cur), to_np(prev)
    ws = ws_tensor(g.eval_moves_workspace_bytes(cfg))
    # explicit list
    moves = gen.explicit_moves(w, 3000, DEV)
    delta = torch.empty(3000, 5, device=DEV)
    best = torch.empty(cfg.L, dtype=torch.int32, device=DEV)
    g.eval_moves(cfg, cur, prev, A, B, D, delta, moves=moves, M=M, M_scalar=0.75, best_per_layer=best, workspace=ws)
    mv = to_np(moves)
    ref = oracle.move_deltas(curn, prevn, mv, An, Bn, Dn, Mn, 0.75, **kw)
    d = to_np(delta).astype(np.float64)
    _check_deltas(cfg, d, ref, mv, curn, An, Bn, Dn, Mn, 0.75)
    for l in range(cfg.L):                                          # lowest dJ of the layer, lowest index on ties
        idx = np.nonzero((mv[:, 0] == l) & ~np.isnan(d[:, 0]))[0]
        dj = to_np(delta)[idx, 0]
        assert int(best[l].item()) == int(idx[np.argmin(dj)])
    # implicit whole neighbourhood in canonical order
    allmv = oracle.all_pair_moves(cfg.L, cfg.NS)
    n = allmv.shape[0]
    delta = torch.empty(n, 5, device=DEV)
    g.eval_moves(cfg, cur, prev, A, B, D, delta, M=M, M_scalar=0.75, best_per_layer=best, workspace=ws)
    d = to_np(delta).astype(np.float64)
    pick = np.arange(n)                                   # the WHOLE neighbourhood (v3 shape: 82,656 moves, ~2 s of oracle)
    ref = oracle.move_deltas(curn, prevn, allmv[pick], An, Bn, Dn, Mn, 0.75, **kw)
    _check_deltas(cfg, d[pick], ref, allmv[pick], curn, An, Bn, Dn, Mn, 0.75)
    per = n // cfg.L
    for l in range(cfg.L):
        seg = to_np(delta)[l * per:(l + 1) * per, 0]
        assert int(best[l].item()) == l * per + int(np.nanargmin(seg))
    # swap deltas equal full re-evaluation through the batched objective as well (BASELINE.json invariant)
    some = pick[~np.isnan(d[pick, 0])][:32]
    cands = cur.unsqueeze(0).repeat(len(some) + 1, 1, 1).contiguous()
    for i, m in enumerate(some):
        l, a, b = allmv[m]
        cands[i + 1, l, a], cands[i + 1, l, b] = cur[l, b], cur[l, a]
    out = torch.empty(len(some) + 1, 5, device=DEV)
    ws2 = ws_tensor(g.eval_placements_workspace_bytes(cfg, len(some) + 1))
    g.eval_placements(cfg, cands, A, B, D, prev, out, M=M, M_scalar=0.75, workspace=ws2)
    o = to_np(out).astype(np.float64)
    full = o[1:] - o[0]
    for j in (1, 2, 3, 4):
        np.testing.assert_allclose(full[:, j], d[some, j], rtol=0, atol=2e-5 * np.abs(o[:, j]).max())


def test_eval_moves_invalid_and_zero_moves():
    w, cfg, A, B, D, M, prev = _placement_instance("v3", 3)
    cur = prev.clone()
    curn = to_np(cur)
    sp = cfg.slots_per_rank
    row = curn[0]
    vals, cnt = np.unique(row, return_counts=True)
    e = vals[cnt == 2][0]
    j0, j1 = np.nonzero(row == e)[0]
    other = (j0 // sp) * sp + ((j0 % sp) + 1) % sp            # a different expert on j0's rank
    moves = torch.tensor([[0, j0, j1],                        # two replicas of one expert: zeros
                          [0, other, j1],                     # would co-locate both copies of e on j0's rank: NaN
                          [0, j0, other],                     # same rank: zeros
                          [1, 0, cfg.NS - 1]], dtype=torch.int32, device=DEV)
    delta = torch.empty(4, 5, device=DEV)
    ws = ws_tensor(g.eval_moves_workspace_bytes(cfg))
    g.eval_moves(cfg, cur, prev, A, B, D, delta, moves=moves, workspace=ws)
    d = to_np(delta)
    ref = oracle.move_deltas(curn, to_np(prev), to_np(moves), to_np(A), to_np(B), to_np(D), None, 1.0, **_oracle_kw(cfg))
    assert np.all(d[0] == 0) and np.all(d[2] == 0) and np.isnan(d[1]).all()
    assert np.array_equal(np.isnan(d), np.isnan(ref))
    # a swap applied twice returns to the start: delta(back) = -delta(forth)
    nxt = cur.clone(); nxt[1, 0], nxt[1, cfg.NS - 1] = cur[1, cfg.NS - 1], cur[1, 0]
    back = torch.empty(1, 5, device=DEV)
    g.eval_moves(cfg, nxt, prev, A, B, D, back, moves=moves[3:4], workspace=ws)
    if not np.isnan(d[3]).any():
        np.testing.assert_allclose(to_np(back)[0, 1:4], -d[3, 1:4], rtol=1e-5, atol=1e-3)


# ------------------------------------------------------------------------------------------
# stats side (a1..a5)
# ------------------------------------------------------------------------------------------
def _router_inputs(w, step=0):
    hidden = gen.hidden_all(w, step, DEV)
    W = gen.w_router(w, DEV)
    slb = gen.src_logit_bias(w, step, DEV)
    sb = gen.select_bias(w, DEV)
    off = gen.src_offsets(w, step, w.T, DEV)
    return hidden, W, slb, sb, off


def _synthetic_logits(w, seed):
    """fp32 logits with the workload's skew plus edge rows: exact ties, NaN, -inf, -0."""
    r = w.router
    gen_ = torch.Generator(device=DEV); gen_.manual_seed(seed)
    x = torch.randn(r.L, w.T, r.E, generator=gen_, device=DEV) * 1.7
    off = gen.src_offsets(w, 0, w.T, DEV)
    slb = gen.src_logit_bias(w, 0, DEV)
    src = torch.repeat_interleave(torch.arange(r.S, device=DEV), (off[1:] - off[:-1]).long())
    x = x + slb[:, src, :]
    x[:, 0::7] = torch.round(x[:, 0::7] * 2) / 2            # many exact ties
    x[:, 5, :] = 0.25                                       # all equal
    x[:, 6, :] = float("-inf")
    x[:, 7, 3] = float("nan")
    x[:, 8, :4] = torch.tensor([0.0, -0.0, 0.0, -0.0], device=DEV)
    x[:, 9, 1] = float("inf")
    return x.contiguous(), off


@pytest.mark.parametrize("name", list(SHAPES))
def test_gating_and_histogram_bit_exact_on_given_logits(name):
    w = _wl(name)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    x, off = _synthetic_logits(w, 11)
    sb = gen.select_bias(w, DEV)
    st = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    ids = torch.full((r.L, w.T, r.k), -9, dtype=torch.int32, device=DEV)
    wts = torch.full((r.L, w.T, r.k), -9.0, device=DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    g.route_stats(cfg, st, T=w.T, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x, topk_ids=ids, topk_w=wts,
                  workspace=ws)
    torch.cuda.synchronize()
    xn, offn = to_np(x), to_np(off)
    for l in range(r.L):
        rid, rw = oracle.gate(xn[l], r, None if sb is None else to_np(sb)[l], tier=1)
        np.testing.assert_array_equal(to_np(ids[l]), rid)                      # bit-exact ids, best first
        finite = np.isfinite(rw).all(1)
        np.testing.assert_allclose(to_np(wts[l])[finite], rw[finite], rtol=1e-5, atol=1e-30)
        C = oracle.counts(rid, offn, r.S, r.E)
        np.testing.assert_array_equal(to_np(st.A_step[l]), C)                  # bit-exact counts
        np.testing.assert_array_equal(C.sum(1), np.diff(offn) * r.k)           # row sums = tokens x k
        if r.n_groups > 1:
            assert all(len(set((row // 32).tolist())) <= r.topk_groups for row in to_np(ids[l]))
    # without the optional outputs the counts are the same
    st2 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    g.route_stats(cfg, st2, T=w.T, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x, workspace=ws)
    assert torch.equal(st2.A_step, st.A_step)


@pytest.mark.parametrize("name,mode", [("v2lite", MODE_EMA), ("qwen3", MODE_WINDOW), ("v3", MODE_WINDOW), ("decode", MODE_EMA)])
def test_update_load_and_pressure_over_steps(name, mode):
    w = _wl(name)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    window_len, decay, steps = 3, 0.9, 7
    st = g.StatsState(cfg, mode, window_len=window_len, ema_decay=decay)
    rng = np.random.default_rng(3)
    Bsyn = rng.integers(1, 1000, (r.L, r.E))
    place = gen.prev_placement(w, Bsyn, DEV)
    dp = gen.dp_of_rank(w, DEV)
    sb = gen.select_bias(w, DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    A_win = np.zeros((r.L, r.S, r.E), np.int64); A_pub = np.zeros_like(A_win); A_ema = np.zeros((r.L, r.S, r.E))
    for step in range(steps):
        x, off = _synthetic_logits(w, 100 + step)
        g.route_stats(cfg, st, T=w.T, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x,
                      cur_placement=place, dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws)
        torch.cuda.synchronize()
        Cs = np.stack([oracle.counts(oracle.gate(to_np(x[l]), r, None if sb is None else to_np(sb)[l], 1)[0], to_np(off), r.S, r.E)
                       for l in range(r.L)])
        np.testing.assert_array_equal(to_np(st.A_step), Cs)
        if mode == MODE_WINDOW:
            live = A_win + Cs                                   # profile after accumulation, before any reset
            pub = oracle.update_window(A_win, Cs, A_pub, step, window_len)
            np.testing.assert_array_equal(to_np(st.A_win), A_win)
            np.testing.assert_array_equal(to_np(st.A_pub), A_pub)
            assert pub == ((step + 1) % window_len == 0)
            d = oracle.derived(live.astype(np.float64), to_np(place), to_np(dp), w.G, w.slots_per_rank)
            np.testing.assert_array_equal(to_np(st.B), d["B"].astype(np.int64))
            if pub:
                np.testing.assert_array_equal(to_np(st.B_pub), d["B"].astype(np.int64))
        else:
            oracle.update_ema(A_ema, Cs, decay)
            np.testing.assert_allclose(to_np(st.A_ema), A_ema, rtol=1e-5)
            d = oracle.derived(A_ema, to_np(place), to_np(dp), w.G, w.slots_per_rank)
            np.testing.assert_allclose(to_np(st.B), d["B"], rtol=1e-5)
        np.testing.assert_allclose(to_np(st.pressure_raw), d["pressure_raw"], rtol=1e-5)
        np.testing.assert_allclose(to_np(st.pressure_rel), d["pressure_rel"], rtol=1e-5)
        np.testing.assert_allclose(to_np(st.pressure_raw).sum(), d["B"].sum(), rtol=1e-5)
        assert int(st.step_counter.item()) == step + 1 and int(st.status.item()) == 0


def _logit_err(gl, rl):
    """|g - r| <= tol * max(|r|, rms(row r)); returns the max of err / that scale."""
    rms = np.sqrt((rl.astype(np.float64) ** 2).mean(-1, keepdims=True))
    return float((np.abs(gl.astype(np.float64) - rl) / np.maximum(np.abs(rl), rms)).max())


@pytest.mark.parametrize("cta_group", [1, 2])
@pytest.mark.parametrize("name", list(SHAPES))
def test_router_gemm_logits_and_full_path(name, cta_group):
    """a1 against the fp64 oracle, then the fused path against (logits OUT -> gating IN)."""
    g.set_option(g.OPT_CTA_GROUP, cta_group)
    w = _wl(name)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    hidden, W, slb, sb, off = _router_inputs(w)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    st = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    logits = torch.full((r.L, w.T, r.E), 7.0, device=DEV)
    ids = torch.full((r.L, w.T, r.k), -9, dtype=torch.int32, device=DEV)
    wts = torch.zeros(r.L, w.T, r.k, device=DEV)
    g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                  logits_mode=g.LOGITS_OUT, logits=logits, topk_ids=ids, topk_w=wts, workspace=ws)
    torch.cuda.synchronize()
    hb, wb, offn = bf16_bits(hidden), bf16_bits(W), to_np(off)
    flips = 0
    for l in range(r.L):
        l64, l32 = oracle.router_logits(hb[l], wb[l], to_np(slb)[l], offn)
        assert _logit_err(to_np(logits[l]), l64) < 1e-2                         # the stated bar
        assert _logit_err(to_np(logits[l]), l64) < 2e-4                         # what fp32 accumulation should give
        # same logits -> same ids / counts, bit-exact
        rid, rw = oracle.gate(to_np(logits[l]), r, None if sb is None else to_np(sb)[l], 1)
        np.testing.assert_array_equal(to_np(ids[l]), rid)
        np.testing.assert_allclose(to_np(wts[l]), rw, rtol=1e-5)
        np.testing.assert_array_equal(to_np(st.A_step[l]), oracle.counts(rid, offn, r.S, r.E))
        # end to end (oracle logits in fp64 -> fp32): report the flip rate
        eid, _ = oracle.gate(l32, r, None if sb is None else to_np(sb)[l], 1)
        flips += int((np.sort(eid, 1) != np.sort(to_np(ids[l]), 1)).any(1).sum())
    rate = flips / (r.L * w.T)
    print(f"[{name} cg{cta_group}] end-to-end top-k flip rate {rate:.2e}")
    assert rate < 5e-3
    # fused, logits never written: identical integers
    st2 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    ids2 = torch.full_like(ids, -9)
    g.route_stats(cfg, st2, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                  logits_mode=g.LOGITS_NONE, topk_ids=ids2, workspace=ws)
    assert torch.equal(ids2, ids) and torch.equal(st2.A_step, st.A_step)
    # counts only, one and two epilogue warps per TMEM lane quadrant (GIMBAL_OPT_EPI_PARTS; two only exists for E >= 128)
    for parts in (1, 2):
        g.set_option(g.OPT_EPI_PARTS, parts)
        st5 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
        g.route_stats(cfg, st5, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off, workspace=ws)
        assert torch.equal(st5.A_step, st.A_step), f"epilogue parts = {parts}"
    g.set_option(g.OPT_EPI_PARTS, 0)
    # unfused two-kernel path (GEMM -> logits -> gating kernel): identical integers again
    g.set_option(g.OPT_FUSE_GATE, 0)
    st3 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    ids3 = torch.full_like(ids, -9)
    logits3 = torch.empty_like(logits)
    g.route_stats(cfg, st3, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                  logits_mode=g.LOGITS_OUT, logits=logits3, topk_ids=ids3, workspace=ws)
    assert torch.equal(logits3, logits) and torch.equal(ids3, ids) and torch.equal(st3.A_step, st.A_step)
    # layer slices give the same result as one call
    if r.L > 1:
        g.set_option(g.OPT_FUSE_GATE, 1)
        st4 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
        for l in range(r.L):
            g.route_stats(cfg, st4, T=w.T, hidden=hidden[l:l + 1], w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                          layer0=l, n_layers=1, workspace=ws)
        assert torch.equal(st4.A_step, st.A_step) and int(st4.step_counter.item()) == 1


def test_gemm_special_cases():
    """one-hot W rows return columns of hidden exactly; all-ones give H; T smaller than a tile."""
    cfg = g.RouterCfg(L=1, H=256, E=16, k=2, S=1)
    T = 37
    hidden = torch.randn(1, T, 256, device=DEV).to(torch.bfloat16)
    W = torch.zeros(1, 16, 256, device=DEV, dtype=torch.bfloat16)
    cols = [7, 0, 255, 64, 63, 128, 1, 2, 3, 4, 5, 6, 8, 9, 10, 11]
    for e, c in enumerate(cols):
        W[0, e, c] = 1.0
    off = torch.tensor([0, T], dtype=torch.int32, device=DEV)
    st = g.StatsState(cfg, MODE_WINDOW)
    logits = torch.empty(1, T, 16, device=DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, 1, T))
    for cg in (1, 2):
        g.set_option(g.OPT_CTA_GROUP, cg)
        logits.fill_(-1)
        g.route_stats(cfg, st, T=T, hidden=hidden, w_router=W, src_offsets=off, logits_mode=g.LOGITS_OUT, logits=logits, workspace=ws)
        assert torch.equal(logits[0], hidden[0][:, cols].float())
        g.route_stats(cfg, st, T=T, hidden=torch.ones_like(hidden), w_router=torch.ones_like(W), src_offsets=off,
                      logits_mode=g.LOGITS_OUT, logits=logits, workspace=ws)
        assert torch.all(logits == 256.0)
    g.set_option(g.OPT_CTA_GROUP, 0)


# ------------------------------------------------------------------------------------------
# NEXT-1: greedy placement heuristic -- integer output, bit-exact
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,counts,table_M,seeded_D", [
    ("tiny", "i32", False, False), ("v2lite", "f32", True, True), ("qwen3", "i32", False, True),
    ("v3", "i32", False, False), ("v3", "f32", True, True), ("decode", "f32", False, False), ("decode", "i32", True, True),
])
def test_greedy_place_parity(name, counts, table_M, seeded_D):
    w, cfg, A, B, D, M, prev = _placement_instance(name, 4, counts, table_M, seeded_D)
    out = torch.full_like(prev, -7)
    status = torch.zeros(1, dtype=torch.int32, device=DEV)
    g.greedy_place(cfg, A, B, D, prev, out, M=M, M_scalar=1.25, status=status)
    torch.cuda.synchronize()
    # the cfg carries the weights as fp32: the oracle gets exactly those values
    wts = tuple(float(np.float32(x)) for x in (cfg.alpha, cfg.beta, cfg.gamma))
    ok, ref = oracle.greedy_place(to_np(prev), to_np(A), to_np(B), to_np(D), to_np(M), 1.25, G=cfg.G, sp=cfg.slots_per_rank, weights=wts)
    np.testing.assert_array_equal(to_np(out), ref)                       # bit-exact placement, failed layers (-1) included
    assert bool(status.item() & 2) == (not ok)
    good = (ref >= 0).all(1)
    assert good.any()
    for l in np.nonzero(good)[0]:                                        # valid placement with x0's expert copies
        assert sorted(ref[l].tolist()) == sorted(to_np(prev)[l].tolist())
    # the result scores through a6 like any candidate (valid: no NaN)
    if good.all():
        cands = torch.stack([prev, out]).contiguous()
        sc = torch.empty(2, 5, device=DEV)
        ws = ws_tensor(g.eval_placements_workspace_bytes(cfg, 2))
        g.eval_placements(cfg, cands, A, B, D, prev, sc, M=M, M_scalar=1.25, workspace=ws)
        s = to_np(sc)
        assert not np.isnan(s).any()


def test_greedy_place_invalid_x0_and_other_weights():
    w, cfg, A, B, D, M, prev = _placement_instance("v3", 5)
    bad = prev.clone(); bad[1, 0] = bad[1, 1]
    out = torch.zeros_like(prev)
    status = torch.zeros(1, dtype=torch.int32, device=DEV)
    g.greedy_place(cfg, A, B, D, bad, out, status=status)
    ok, ref = oracle.greedy_place(to_np(bad), to_np(A), to_np(B), to_np(D), None, 1.0, G=cfg.G, sp=cfg.slots_per_rank,
                                  weights=tuple(float(np.float32(x)) for x in (cfg.alpha, cfg.beta, cfg.gamma)))
    assert not ok and (ref[1] == -1).all()
    np.testing.assert_array_equal(to_np(out), ref)
    assert int(status.item()) & 2
    for wts in [(1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 0.0), (1.0, 0.0025, 1e9)]:
        cfg2 = g.PlacementCfg(L=cfg.L, E=cfg.E, G=cfg.G, slots_per_rank=cfg.slots_per_rank, S=cfg.S, alpha=wts[0], beta=wts[1], gamma=wts[2])
        g.greedy_place(cfg2, A, B, D, prev, out)
        ok, ref = oracle.greedy_place(to_np(prev), to_np(A), to_np(B), to_np(D), None, 1.0, G=cfg.G, sp=cfg.slots_per_rank,
                                      weights=tuple(float(np.float32(x)) for x in wts))
        np.testing.assert_array_equal(to_np(out), ref)


# ------------------------------------------------------------------------------------------
# NEXT-3: logical -> physical expert mapping fused with counting (R18)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(SHAPES))
@pytest.mark.parametrize("mode", ["logits_in", "fused"])
def test_expert_mapping_parity(name, mode):
    w = _wl(name)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    rng = np.random.default_rng(12)
    place = gen.prev_placement(w, rng.integers(1, 1000, (r.L, r.E)), DEV)
    status = torch.zeros(1, dtype=torch.int32, device=DEV)
    emap = g.ExpertMap(r.L, r.E, w.G, w.slots_per_rank, place, status=status)
    st = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    ids = torch.full((r.L, w.T, r.k), -9, dtype=torch.int32, device=DEV)
    phys = torch.full((r.L, w.T, r.k), -9, dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    sb = gen.select_bias(w, DEV)
    if mode == "logits_in":
        x, off = _synthetic_logits(w, 21)
        g.route_stats(cfg, st, T=w.T, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x, topk_ids=ids,
                      expert_map=emap, phys_ids=phys, workspace=ws)
    else:
        hidden, W, slb, sb, off = _router_inputs(w)
        g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                      topk_ids=ids, expert_map=emap, phys_ids=phys, workspace=ws)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    pl = to_np(place)
    for l in range(r.L):
        ref = oracle.expert_map(to_np(ids[l]), pl[l])
        np.testing.assert_array_equal(to_np(phys[l]), ref)                   # bit-exact slots
        assert (pl[l][ref] == to_np(ids[l])).all()                           # every slot hosts the chosen expert
        # the inverse tables themselves: slots grouped by expert, ascending inside a group
        off_l, slots_l = to_np(emap.rep_off[l]), to_np(emap.rep_slots[l])
        for e in range(r.E):
            np.testing.assert_array_equal(slots_l[off_l[e]:off_l[e + 1]], np.nonzero(pl[l] == e)[0])
    # the mapping does not disturb the counts; without topk_ids the same slots come out
    st2 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    phys2 = torch.full_like(phys, -9)
    if mode == "logits_in":
        g.route_stats(cfg, st2, T=w.T, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x, expert_map=emap,
                      phys_ids=phys2, workspace=ws)
    else:
        g.route_stats(cfg, st2, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                      expert_map=emap, phys_ids=phys2, workspace=ws)
    assert torch.equal(phys2, phys) and torch.equal(st2.A_step, st.A_step)


# ------------------------------------------------------------------------------------------
# the calls are asynchronous, allocation-free and capturable in a CUDA graph (include/gimbal.h conventions)
# ------------------------------------------------------------------------------------------
def test_cuda_graph_capture_of_a_whole_step():
    w = _wl("decode")
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    hidden, W, slb, sb, off = _router_inputs(w)
    dp = gen.dp_of_rank(w, DEV)
    pc = g.PlacementCfg(L=r.L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S, counts_dtype=g.COUNTS_F32)
    prev = gen.prev_placement(w, np.ones((r.L, r.E)), DEV)
    cands = gen.candidates(w, prev, w.P, DEV)
    D = gen.comm_cost_D(w, "binary", DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    wsp = ws_tensor(g.eval_placements_workspace_bytes(pc, w.P))
    n = r.L * w.NS * (w.NS - 1) // 2

    def make():
        st = g.StatsState(cfg, MODE_EMA, ema_decay=0.9)
        return st, torch.zeros(w.P, 5, device=DEV), torch.zeros(n, 5, device=DEV), torch.zeros(r.L, dtype=torch.int32, device=DEV), \
            torch.zeros_like(prev)

    def step(st, out, delta, best, greedy, stream=None):
        g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                      cur_placement=prev, dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws, stream=stream)
        g.eval_placements(pc, cands, st.A_ema, st.B, D, prev, out, workspace=wsp, stream=stream)
        g.eval_moves(pc, prev, prev, st.A_ema, st.B, D, delta, best_per_layer=best, workspace=wsp, stream=stream)
        g.greedy_place(pc, st.A_ema, st.B, D, prev, greedy, stream=stream)

    g.kernel_timing(False)                        # event brackets must be off while capturing
    # eager: three steps
    ref = make()
    for _ in range(3):
        step(*ref)
    torch.cuda.synchronize()
    # captured once, replayed three times on fresh state
    cap = make()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step(*cap, stream=side)                   # warm-up outside the capture (function attributes, module load)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    for t in (cap[0].A_ema, cap[0].B, cap[0].step_counter, cap[0].A_step):
        t.zero_()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        step(*cap, stream=side)
    for t in (cap[0].A_ema, cap[0].B, cap[0].step_counter, cap[0].A_step):
        t.zero_()                                 # the capture itself ran nothing; start from the initial state
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    assert int(cap[0].step_counter.item()) == 3 == int(ref[0].step_counter.item())
    assert torch.equal(cap[0].A_ema, ref[0].A_ema) and torch.equal(cap[0].B, ref[0].B)
    assert torch.equal(cap[1], ref[1]) and torch.equal(cap[3], ref[3]) and torch.equal(cap[4], ref[4])
    assert torch.equal(torch.nan_to_num(cap[2]), torch.nan_to_num(ref[2]))


# ------------------------------------------------------------------------------------------
# gating variants that no BASELINE.json config exercises (E = 32, grouped softmax, ungrouped sigmoid, topn = 1, k < 8)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("E,k,score_fn,renorm,n_groups,topk_groups,topn,bias", [
    (32, 4, 0, 0, 1, 1, 1, False),
    (16, 1, 1, 0, 1, 1, 1, True),
    (64, 3, 1, 1, 1, 1, 1, True),
    (64, 8, 0, 1, 2, 1, 2, False),
    (128, 5, 0, 0, 4, 2, 1, False),
    (256, 3, 1, 0, 8, 3, 1, False),
    (256, 8, 1, 1, 8, 2, 2, True),
])
def test_gating_variants(E, k, score_fn, renorm, n_groups, topk_groups, topn, bias):
    from workloads.configs import RouterCfg as WRouterCfg
    L, T, S, H = 2, 700, 3, 128
    r = WRouterCfg(L=L, H=H, E=E, k=k, S=S, score_fn=score_fn, renorm=renorm, n_groups=n_groups, topk_groups=topk_groups,
                   group_score_topn=topn, routed_scale=1.5)
    cfg = g.RouterCfg.from_workload(r)
    gen_ = torch.Generator(device=DEV); gen_.manual_seed(E * 100 + k)
    x = torch.randn(L, T, E, generator=gen_, device=DEV) * 2.0
    x[:, 0::5] = torch.round(x[:, 0::5] * 2) / 2                           # many exact ties
    x[:, 3, :] = -1.0                                                       # an all-equal row
    off = torch.tensor([0, 250, 250, T], dtype=torch.int32, device=DEV)     # one empty source
    sb = (0.05 * torch.randn(L, E, generator=gen_, device=DEV)) if bias else None
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, L, T))

    def check(ids, wts, st, logits):
        for l in range(L):
            rid, rw = oracle.gate(to_np(logits[l]), r, None if sb is None else to_np(sb)[l], tier=1)
            np.testing.assert_array_equal(to_np(ids[l]), rid)
            np.testing.assert_allclose(to_np(wts[l]), rw, rtol=1e-5, atol=1e-30)
            np.testing.assert_array_equal(to_np(st.A_step[l]), oracle.counts(rid, to_np(off), S, E))

    # standalone kernel: with outputs (one lane per row) and without (R lanes per row) must agree with the oracle
    st = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    ids = torch.full((L, T, k), -9, dtype=torch.int32, device=DEV)
    wts = torch.full((L, T, k), -9.0, device=DEV)
    g.route_stats(cfg, st, T=T, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x, topk_ids=ids, topk_w=wts, workspace=ws)
    check(ids, wts, st, x)
    st2 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    g.route_stats(cfg, st2, T=T, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x, workspace=ws)
    assert torch.equal(st2.A_step, st.A_step)
    # fused GEMM epilogue on its own logits
    hidden = torch.randn(L, T, H, generator=gen_, device=DEV).to(torch.bfloat16)
    W = (0.2 * torch.randn(L, E, H, generator=gen_, device=DEV)).to(torch.bfloat16)
    for cg in (1, 2):
        g.set_option(g.OPT_CTA_GROUP, cg)
        st3 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
        logits = torch.empty(L, T, E, device=DEV)
        g.route_stats(cfg, st3, T=T, hidden=hidden, w_router=W, select_bias=sb, src_offsets=off, logits_mode=g.LOGITS_OUT, logits=logits,
                      topk_ids=ids, topk_w=wts, workspace=ws)
        check(ids, wts, st3, logits)
        st4 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
        g.route_stats(cfg, st4, T=T, hidden=hidden, w_router=W, select_bias=sb, src_offsets=off, workspace=ws)
        assert torch.equal(st4.A_step, st3.A_step)
    g.set_option(g.OPT_CTA_GROUP, 0)


def test_route_stats_edges_empty_step_and_many_sources():
    """T = 0 (an idle step still advances the window / EMA) and S = 64 sources with E = 256 (the largest histogram)."""
    from workloads.configs import RouterCfg as WRouterCfg
    r = WRouterCfg(L=2, H=128, E=256, k=8, S=64, score_fn=1, renorm=1, n_groups=8, topk_groups=4, group_score_topn=2, routed_scale=2.5)
    cfg = g.RouterCfg.from_workload(r)
    T = 900
    gen_ = torch.Generator(device=DEV); gen_.manual_seed(3)
    hidden = torch.randn(r.L, T, r.H, generator=gen_, device=DEV).to(torch.bfloat16)
    W = (0.3 * torch.randn(r.L, r.E, r.H, generator=gen_, device=DEV)).to(torch.bfloat16)
    cuts = np.sort(np.random.default_rng(1).integers(0, T + 1, r.S - 1))
    off = torch.from_numpy(np.concatenate([[0], cuts, [T]]).astype(np.int32)).to(DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, T))
    st = g.StatsState(cfg, MODE_EMA, ema_decay=0.5)
    logits = torch.empty(r.L, T, r.E, device=DEV)
    ids = torch.empty(r.L, T, r.k, dtype=torch.int32, device=DEV)
    g.route_stats(cfg, st, T=T, hidden=hidden, w_router=W, src_offsets=off, logits_mode=g.LOGITS_OUT, logits=logits, topk_ids=ids, workspace=ws)
    st_f = g.StatsState(cfg, MODE_EMA, ema_decay=0.5)
    g.route_stats(cfg, st_f, T=T, hidden=hidden, w_router=W, src_offsets=off, workspace=ws)     # fused, nothing written
    for l in range(r.L):
        rid, _ = oracle.gate(to_np(logits[l]), r, None, 1)
        np.testing.assert_array_equal(to_np(ids[l]), rid)
        np.testing.assert_array_equal(to_np(st.A_step[l]), oracle.counts(rid, to_np(off), r.S, r.E))
    assert torch.equal(st_f.A_step, st.A_step) and torch.equal(st_f.A_ema, st.A_ema)
    # an empty step: counts are zero, the EMA decays, the step counter advances
    before = st.A_ema.clone()
    off0 = torch.zeros(r.S + 1, dtype=torch.int32, device=DEV)
    g.route_stats(cfg, st, T=0, hidden=hidden, w_router=W, src_offsets=off0, workspace=ws)
    assert int(st.A_step.abs().sum().item()) == 0 and int(st.step_counter.item()) == 2
    assert torch.equal(st.A_ema, before * 0.5)


# ------------------------------------------------------------------------------------------
# NEXT-2: Algorithm 1, Global DP Engine Scheduling (R19) -- integer output, bit-exact
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,R,params", [
    (2, 40, dict()),
    (8, 64, dict(lambda_kv=200.0, lambda_moe=150.0, close_frac=0.25)),
    (16, 50, dict(lambda_kv=50.0, lambda_moe=500.0, close_frac=0.05)),
    (33, 30, dict(lambda_moe=80.0)),
    (64, 70, dict(lambda_kv=10.0, lambda_moe=10.0, close_frac=1.0)),
])
def test_select_engines_parity(N, R, params):
    rng = np.random.default_rng(N * 7 + R)
    B = 1500
    tr = np.stack([rng.uniform(0.05, 0.99, (B, N)), rng.integers(0, 4000, (B, N)), rng.integers(0, 2000, (B, N)),
                   rng.uniform(0.3, 2.0, (B, N))], -1).astype(np.float32)
    tr[::5, :, 0] = rng.uniform(0.05, 0.85, (len(tr[::5]), N))            # instances where the KV rule cannot fire
    tr[1::7, :, 1:3] = 100.0                                              # equal pressure: ties / CLOSE decide
    lens = np.ceil(rng.lognormal(6.0, 1.0, (B, R))).astype(np.float32)
    complete = (rng.random(B) > 0.1).astype(np.uint8)
    rr0 = rng.integers(0, N, B).astype(np.int32)
    comp0 = rng.integers(0, 500, (B, N)).astype(np.float64)
    t = lambda a: torch.from_numpy(a).to(DEV)
    comp, rr, eng = t(comp0.copy()), t(rr0.copy()), torch.full((B, R), -3, dtype=torch.int32, device=DEV)
    g.select_engines(t(tr), t(lens), comp, rr, eng, complete=t(complete), **params)
    torch.cuda.synchronize()
    p32 = {k: float(np.float32(v)) for k, v in params.items()}            # the C struct carries fp32 parameters
    p32.setdefault("high_kv", float(np.float32(0.9))); p32.setdefault("large_gap", float(np.float32(0.1)))
    ge, gc, gr = to_np(eng), to_np(comp), to_np(rr)
    for b in range(0, B, 3):
        c = comp0[b].copy()
        e, r_after = oracle.select_engines(tr[b], complete[b], lens[b], c, rr0[b], **p32)
        np.testing.assert_array_equal(ge[b], e)
        np.testing.assert_array_equal(gc[b], c)
        assert gr[b] == r_after
    assert ((ge >= 0) & (ge < N)).all()
    np.testing.assert_allclose(gc.sum(1), comp0.sum(1) + lens.astype(np.float64).sum(1), rtol=1e-12)   # every request is assigned once


def test_select_engines_consumes_route_stats_pressure():
    """the loop the paper closes: pressure_rel of the stats path is the moe column of the trace"""
    w = _wl("qwen3")
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    x, off = _synthetic_logits(w, 31)
    place = gen.prev_placement(w, np.random.default_rng(2).integers(1, 1000, (r.L, r.E)), DEV)
    dp = gen.dp_of_rank(w, DEV)
    st = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    g.route_stats(cfg, st, T=w.T, src_offsets=off, logits_mode=g.LOGITS_IN, logits=x, cur_placement=place, dp_of_rank=dp, G=w.G,
                  slots_per_rank=w.slots_per_rank, workspace=ws)
    N, R = r.S, 32
    tr = torch.zeros(1, N, 4, device=DEV)
    tr[0, :, 0] = 0.5; tr[0, :, 1] = 1000.0; tr[0, :, 3] = st.pressure_rel
    lens = torch.full((1, R), 10.0, device=DEV)
    comp = torch.zeros(1, N, dtype=torch.float64, device=DEV); rr = torch.zeros(1, dtype=torch.int32, device=DEV)
    eng = torch.empty(1, R, dtype=torch.int32, device=DEV)
    g.select_engines(tr, lens, comp, rr, eng, lambda_moe=1000.0)
    c = np.zeros(N)
    e, _ = oracle.select_engines(to_np(tr)[0], 1, to_np(lens)[0], c, 0, lambda_moe=1000.0)
    np.testing.assert_array_equal(to_np(eng)[0], e)
    assert int(to_np(eng)[0, 0]) == int(np.argmin(to_np(st.pressure_rel)))       # the engine with the least MoE pressure goes first


# ------------------------------------------------------------------------------------------
# Algorithm 2, SJF with aging (R20) -- a permutation, bit-exact
# ------------------------------------------------------------------------------------------
def test_order_queues_parity():
    rng = np.random.default_rng(17)
    B, Q = 300, 700
    arrival = rng.uniform(0, 20, (B, Q)).round(1).astype(np.float32)
    prefill = np.ceil(rng.lognormal(5.0, 1.2, (B, Q))).astype(np.int32)
    prefill[:, ::9] = 64                                                  # equal lengths
    qlen = rng.integers(0, Q + 1, B).astype(np.int32)
    qlen[:3] = [0, 1, Q]
    now, theta = 20.0, 5.0
    t = lambda a: torch.from_numpy(a).to(DEV)
    order = torch.full((B, Q), -5, dtype=torch.int32, device=DEV)
    g.order_queues(t(arrival), t(prefill), t(qlen), now, order, theta_age=theta)
    torch.cuda.synchronize()
    go = to_np(order)
    for b in range(B):
        n = int(qlen[b])
        np.testing.assert_array_equal(go[b, :n], oracle.order_queue(arrival[b, :n], prefill[b, :n], now, theta))
        assert (go[b, n:] == -1).all()


# ------------------------------------------------------------------------------------------
# NEXT-4: calibration sweep of (beta, gamma) against the exhaustive reference (analogue of Fig. 6)
# ------------------------------------------------------------------------------------------
def test_calibration_sweep_against_oracle():
    import math
    from paper_2606_15177_b200 import calibrate
    rng = np.random.default_rng(21)
    n, S, E, G, sp = 6, 2, 8, 4, 2
    A = rng.integers(0, 400, (n, S, E))
    A[:, 0, :E // 2] += 300; A[:, 1, E // 2:] += 300                    # source-dependent skew
    B = A.sum(1)
    D = (np.arange(G)[None, :] * S // G != np.arange(S)[:, None]).astype(np.float32)
    prev = np.stack([rng.permutation(E) for _ in range(n)]).astype(np.int16)
    betas, gammas = [0.0, 0.0025, 0.05], [0.0, 1.0, 100.0]
    res = calibrate.calibration_sweep(A, B, D, prev, G, sp, betas, gammas, device=DEV)
    assert calibrate.all_placements(E, G, sp).shape[0] == math.factorial(E) // math.factorial(sp) ** G == 2520
    Af, Bf = A.astype(np.float64), B.astype(np.float64)
    for i in range(n):      # the reference is a minimiser of the printed objective (weights 1,1,1): same J as the oracle's brute force
        cnt, Jopt, _ = oracle.bruteforce(prev[i], Af[i], Bf[i], D, None, 1.0, G=G, sp=sp, weights=(1.0, 1.0, 1.0))
        Jref = oracle.objective(res["ref"][i][None], prev[i][None], Af[i][None], Bf[i][None], D, None, 1.0, G=G, sp=sp, weights=(1.0, 1.0, 1.0))
        assert cnt == 2520 and abs(Jref[0] - Jopt) <= 1e-5 * Jopt
        np.testing.assert_allclose(res["ref_comm"][i], Jref[2], rtol=1e-5)
    # agreement / communication gap recomputed with the oracle's greedy and objective
    for bi, beta in enumerate(betas):
        for gi, gamma in enumerate(gammas):
            wts = tuple(float(np.float32(x)) for x in (1.0, beta, gamma))
            ok, placed = oracle.greedy_place(prev, Af, Bf, D, None, 1.0, G=G, sp=sp, weights=wts)
            assert ok
            same = [float((calibrate.rank_of(placed[i], sp) == calibrate.rank_of(res["ref"][i], sp)).mean()) for i in range(n)]
            comm = [oracle.objective(placed[i][None], prev[i][None], Af[i][None], Bf[i][None], D, None, 1.0, G=G, sp=sp)[2] for i in range(n)]
            assert abs(res["agree"][bi, gi] - np.mean(same)) < 1e-12
            np.testing.assert_allclose(res["comm_gap"][bi, gi], np.mean(np.array(comm) / res["ref_comm"] - 1.0), rtol=1e-4, atol=1e-6)
    # a prohibitive migration weight freezes the placement at x0: the heuristic then agrees with the reference exactly as much as x0 does
    x0_agree = np.mean([(calibrate.rank_of(prev[i], sp) == calibrate.rank_of(res["ref"][i], sp)).mean() for i in range(n)])
    frozen = calibrate.calibration_sweep(A, B, D, prev, G, sp, [0.0025], [1e9], device=DEV)
    assert abs(frozen["agree"][0, 0] - x0_agree) < 1e-12
    assert res["best"][0] in betas and res["best"][1] in gammas


@pytest.mark.parametrize("H,T,E", [(64, 1, 16), (64, 129, 64), (192, 257, 128), (320, 511, 256), (7168, 130, 256)])
def test_router_gemm_odd_shapes(H, T, E):
    """one k-block, a single token, tiles with ragged tails, both CTA-group modes: logits against the fp64 oracle, counts
    against the oracle on the GPU's logits"""
    from workloads.configs import RouterCfg as WRouterCfg
    L, S, k = 3, 2, min(4, E)
    r = WRouterCfg(L=L, H=H, E=E, k=k, S=S)
    cfg = g.RouterCfg.from_workload(r)
    gen_ = torch.Generator(device=DEV); gen_.manual_seed(H + T + E)
    hidden = torch.randn(L, T, H, generator=gen_, device=DEV).to(torch.bfloat16)
    W = (0.1 * torch.randn(L, E, H, generator=gen_, device=DEV)).to(torch.bfloat16)
    off = torch.tensor([0, T // 3, T], dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, L, T))
    hb, wb, offn = bf16_bits(hidden), bf16_bits(W), to_np(off)
    for cgm in (1, 2):
        g.set_option(g.OPT_CTA_GROUP, cgm)
        st = g.StatsState(cfg, MODE_WINDOW, window_len=1)
        logits = torch.full((L, T, E), 9.0, device=DEV)
        g.route_stats(cfg, st, T=T, hidden=hidden, w_router=W, src_offsets=off, logits_mode=g.LOGITS_OUT, logits=logits, workspace=ws)
        st2 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
        g.route_stats(cfg, st2, T=T, hidden=hidden, w_router=W, src_offsets=off, workspace=ws)
        for l in range(L):
            l64, _ = oracle.router_logits(hb[l], wb[l], None, offn)
            assert _logit_err(to_np(logits[l]), l64) < 2e-4
            rid, _ = oracle.gate(to_np(logits[l]), r, None, 1)
            np.testing.assert_array_equal(to_np(st.A_step[l]), oracle.counts(rid, offn, S, E))
        assert torch.equal(st2.A_step, st.A_step)
    g.set_option(g.OPT_CTA_GROUP, 0)


def test_repeated_launches_are_deterministic():
    """the persistent tcgen05 kernel, its mbarrier pipeline and the histogram flushes give the same integers on every
    launch (a lost arrival or a race would show up as a differing count or a hang)"""
    w = scaled(get_workload("v3"), L=3, T=4100)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    hidden, W, slb, sb, off = _router_inputs(w)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    st = g.StatsState(cfg, MODE_WINDOW, window_len=1000)
    first = None
    for it in range(40):
        g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off, workspace=ws)
        if first is None:
            first = st.A_step.clone()
        else:
            assert torch.equal(st.A_step, first)
    torch.cuda.synchronize()
    assert torch.equal(st.A_win, first * 40) and int(st.step_counter.item()) == 40


# ------------------------------------------------------------------------------------------
# swap-based refinement on top of a7 (R21)
# ------------------------------------------------------------------------------------------
def test_refine_placement_bit_exact_on_integer_instances_and_monotone_elsewhere():
    # (1) integer counts, binary D, M = 1, weights (1,1,1): every delta is an integer that fp32 holds exactly, so the
    # kernel and the fp64 oracle take the same decisions -> identical placements
    rng = np.random.default_rng(41)
    L, S, E, G, sp = 3, 2, 16, 4, 4
    A = rng.integers(0, 60, (L, S, E)); B = A.sum(1)
    D = (np.arange(G)[None, :] * S // G != np.arange(S)[:, None]).astype(np.float32)
    prev = np.stack([rng.permutation(E) for _ in range(L)]).astype(np.int16)
    cfg = g.PlacementCfg(L=L, E=E, G=G, slots_per_rank=sp, S=S, alpha=1.0, beta=1.0, gamma=1.0)
    t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(device=DEV, dtype=dt)
    A_t, B_t, D_t, prev_t = t(A, torch.int32), t(B, torch.int32), t(D, torch.float32), t(prev, torch.int16)
    n = L * (E * (E - 1) // 2)
    delta = torch.empty(n, 5, device=DEV); best = torch.empty(L, dtype=torch.int32, device=DEV)
    applied = torch.full((L,), -1, dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.eval_moves_workspace_bytes(cfg))
    cur = prev_t.clone()
    g.refine_placement(cfg, cur, prev_t, A_t, B_t, D_t, delta, best, iters=12, applied=applied, workspace=ws)
    ref, ref_applied = oracle.refine(prev, prev, A, B, D, None, 1.0, G=G, sp=sp, weights=(1.0, 1.0, 1.0), iters=12)
    np.testing.assert_array_equal(to_np(cur), ref)
    np.testing.assert_array_equal(to_np(applied), ref_applied)
    assert ref_applied.sum() > 0
    # (2) a V3-shaped instance with fp32 counts and an M table: the objective (oracle) never increases from round to round
    w, cfg, A, B, D, M, prev = _placement_instance("v3", 6, "f32", True, True)
    cur = gen.candidates(w, prev, 4, DEV)[3].contiguous()
    n = cfg.L * cfg.NS * (cfg.NS - 1) // 2
    delta = torch.empty(n, 5, device=DEV); best = torch.empty(cfg.L, dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.eval_moves_workspace_bytes(cfg))
    kw = _oracle_kw(cfg)
    J = [oracle.objective(to_np(cur), to_np(prev), to_np(A), to_np(B), to_np(D), to_np(M), 0.75, **kw)[0]]
    for it in range(4):
        g.refine_placement(cfg, cur, prev, A, B, D, delta, best, iters=1, M=M, M_scalar=0.75, workspace=ws)
        J.append(oracle.objective(to_np(cur), to_np(prev), to_np(A), to_np(B), to_np(D), to_np(M), 0.75, **kw)[0])
        assert not np.isnan(J[-1]) and J[-1] <= J[-2] * (1 + 1e-9)
    assert J[-1] < J[0]


# ------------------------------------------------------------------------------------------
# the *_host entry points (bench.py's e2e leg): bit for bit the device-pointer calls
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,n_stage", [("v3", 2), ("v2lite", 3), ("decode", 2)])
def test_host_entry_points_match_device_calls(name, n_stage):
    """gimbal_route_stats_host (layer-sliced calls on the context's copy stream, a 2-slot staging ring under >= 3 layers),
    gimbal_eval_placements_host and gimbal_eval_moves_host against the device-pointer calls on the same inputs: same
    integers, same floats, bit for bit -- over two consecutive steps so that the window / EMA state carries over."""
    w = scaled(get_workload(name), L=4, T=700, P=48)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    W = gen.w_router(w, DEV); sb = gen.select_bias(w, DEV); dp = gen.dp_of_rank(w, DEV)
    place = gen.prev_placement(w, np.random.default_rng(9).integers(1, 1000, (r.L, r.E)), DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    mode = w.mode
    st_d = g.StatsState(cfg, mode, window_len=2, ema_decay=0.9)
    st_h = g.StatsState(cfg, mode, window_len=2, ema_decay=0.9)
    ctx = g.HostCtx()
    layer_bytes = w.T * r.H * 2
    stage = torch.empty(n_stage * layer_bytes, dtype=torch.uint8, device=DEV)
    off_stage = torch.empty(r.S + 1, dtype=torch.int32, device=DEV)
    res = torch.empty(g.route_stats_result_bytes(cfg), dtype=torch.uint8).pin_memory()
    for step in range(2):
        hidden = gen.hidden_all(w, step, DEV)
        slb = gen.src_logit_bias(w, step, DEV)
        off = gen.src_offsets(w, step, w.T, DEV)
        g.route_stats(cfg, st_d, T=w.T, hidden=hidden, w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off,
                      cur_placement=place, dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, workspace=ws)
        hidden_host = hidden.cpu().pin_memory()
        off_host = off.cpu().pin_memory()
        g.route_stats_host(ctx, cfg, st_h, T=w.T, hidden_host=hidden_host, src_offsets_host=off_host, hidden_stage=stage,
                           src_offsets_stage=off_stage, w_router=W, select_bias=sb, src_logit_bias=slb, cur_placement=place,
                           dp_of_rank=dp, G=w.G, slots_per_rank=w.slots_per_rank, result_host=res, workspace=ws)
        torch.cuda.synchronize()
        for a, b in ((st_h.A_step, st_d.A_step), (st_h.A_win, st_d.A_win), (st_h.A_pub, st_d.A_pub), (st_h.A_ema, st_d.A_ema),
                     (st_h.B, st_d.B), (st_h.pressure_raw, st_d.pressure_raw), (st_h.pressure_rel, st_d.pressure_rel),
                     (st_h.step_counter, st_d.step_counter)):
            assert torch.equal(a, b)
        # the result block: A_step i32 [L,S,E] | B [L,E] | pressure_raw [S] | pressure_rel [S]
        nA, nB = 4 * r.L * r.S * r.E, 4 * r.L * r.E
        rb = res.numpy()
        np.testing.assert_array_equal(rb[:nA].view(np.int32).reshape(r.L, r.S, r.E), to_np(st_d.A_step))
        np.testing.assert_array_equal(rb[nA:nA + nB].view(np.int32 if mode == MODE_WINDOW else np.float32).reshape(r.L, r.E), to_np(st_d.B))
        np.testing.assert_array_equal(rb[nA + nB:nA + nB + 4 * r.S].view(np.float32), to_np(st_d.pressure_raw))
        np.testing.assert_array_equal(rb[nA + nB + 4 * r.S:].view(np.float32), to_np(st_d.pressure_rel))
    ctx.close()
    # against the oracle as well: the last step's counts on the host path's own state
    assert int(st_h.status.item()) == 0 and int(st_h.A_step.sum().item()) == r.L * w.T * r.k
    # ---- placements / moves with host buffers
    pc = g.PlacementCfg(L=r.L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S,
                        counts_dtype=g.COUNTS_I32 if mode == MODE_WINDOW else g.COUNTS_F32)
    A_live = st_d.A_step if mode == MODE_WINDOW else st_d.A_ema
    D = gen.comm_cost_D(w, "seeded", DEV)
    cands = gen.candidates(w, place, w.P, DEV)
    wsp = ws_tensor(g.eval_placements_workspace_bytes(pc, w.P))
    out_d = torch.empty(w.P, 5, device=DEV); am_d = torch.zeros(1, dtype=torch.int32, device=DEV)
    g.eval_placements(pc, cands, A_live, st_d.B, D, place, out_d, argmin=am_d, workspace=wsp)
    out_h = torch.empty(w.P, 5).pin_memory(); am_h = torch.zeros(1, dtype=torch.int32).pin_memory()
    g.eval_placements_host(pc, cands.cpu().pin_memory(), torch.empty_like(cands), torch.empty(w.P, 5, device=DEV), A_live, st_d.B, D,
                           place, out_h, argmin_host=am_h, workspace=wsp)
    assert torch.equal(out_h, out_d.cpu()) and int(am_h.item()) == int(am_d.item())
    ref = oracle.objective_batch(to_np(cands), to_np(place), to_np(A_live), to_np(st_d.B), to_np(D), None, 1.0, **_oracle_kw(pc))
    _check_objective(out_h.numpy().astype(np.float64), ref)
    cur = cands[2].contiguous()
    n = r.L * w.NS * (w.NS - 1) // 2
    delta_d = torch.empty(n, 5, device=DEV); best_d = torch.empty(r.L, dtype=torch.int32, device=DEV)
    g.eval_moves(pc, cur, place, A_live, st_d.B, D, delta_d, best_per_layer=best_d, workspace=wsp)
    delta_s = torch.empty(n, 5, device=DEV); best_s = torch.empty(r.L, dtype=torch.int32, device=DEV)
    delta_h = torch.empty(n, 5).pin_memory(); best_h = torch.empty(r.L, dtype=torch.int32).pin_memory()
    g.eval_moves_host(pc, cur.cpu().pin_memory(), place.cpu().pin_memory(), torch.empty_like(cur), torch.empty_like(place), A_live, st_d.B, D,
                      delta_s, delta_host=delta_h, best_stage=best_s, best_host=best_h, workspace=wsp)
    assert torch.equal(torch.nan_to_num(delta_h, nan=-7.0), torch.nan_to_num(delta_d.cpu(), nan=-7.0)) and torch.equal(best_h, best_d.cpu())
    mv = gen.explicit_moves(w, 500, DEV)
    dl_d = torch.empty(500, 5, device=DEV)
    g.eval_moves(pc, cur, place, A_live, st_d.B, D, dl_d, moves=mv, workspace=wsp)
    dl_h = torch.empty(500, 5).pin_memory()
    g.eval_moves_host(pc, cur.cpu().pin_memory(), place.cpu().pin_memory(), torch.empty_like(cur), torch.empty_like(place), A_live, st_d.B, D,
                      torch.empty(500, 5, device=DEV), moves_host=mv.cpu().pin_memory(), moves_stage=torch.empty_like(mv), delta_host=dl_h,
                      workspace=wsp)
    assert torch.equal(torch.nan_to_num(dl_h, nan=-7.0), torch.nan_to_num(dl_d.cpu(), nan=-7.0))


def test_misaligned_bias_is_rejected_on_the_host():
    """the fused epilogue reads a token's src_logit_bias row with 16-byte loads: a 4-byte-aligned view is refused up front
    (INVALID_ARG, nothing launched) instead of trapping on the device"""
    w = _wl("tiny")
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    hidden, W, slb, sb, off = _router_inputs(w)
    buf = torch.zeros(slb.numel() + 1, device=DEV)
    view = buf[1:].view_as(slb)
    view.copy_(slb)
    assert view.data_ptr() % 16 == 4
    st = g.StatsState(cfg, MODE_WINDOW)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    n0 = g.launch_count()
    with pytest.raises(g.GimbalError, match="src_logit_bias must be 16-byte aligned"):
        g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, src_logit_bias=view, src_offsets=off, workspace=ws)
    assert g.launch_count() == n0
    g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, src_logit_bias=slb, src_offsets=off, workspace=ws)
    torch.cuda.synchronize()
    assert int(st.A_step.sum().item()) == r.L * w.T * r.k


def test_scheduler_kernels_on_stale_pointer_and_nan_arrival():
    """Algorithm 1's ordered-dispatch pointer counts modulo N whatever the caller left in it (R19); a NaN arrival time is
    the youngest request in Algorithm 2 (R20) -- both against the oracle, and the order stays a permutation."""
    N, R = 5, 12
    rng = np.random.default_rng(5)
    tr = np.stack([rng.uniform(0.1, 0.5, (4, N)), rng.integers(0, 100, (4, N)), rng.integers(0, 100, (4, N)), np.ones((4, N))], -1).astype(np.float32)
    lens = rng.integers(1, 50, (4, R)).astype(np.float32)
    rr0 = np.array([-7, 13, 5, -1], np.int32)
    complete = np.zeros(4, np.uint8)                                      # incomplete traces: pure ordered dispatch
    t = lambda a: torch.from_numpy(a).to(DEV)
    comp, rr, eng = t(np.zeros((4, N))), t(rr0.copy()), torch.full((4, R), -3, dtype=torch.int32, device=DEV)
    g.select_engines(t(tr), t(lens), comp, rr, eng, complete=t(complete))
    for b in range(4):
        c = np.zeros(N)
        e, r_after = oracle.select_engines(tr[b], 0, lens[b], c, int(rr0[b]))
        np.testing.assert_array_equal(to_np(eng)[b], e)
        assert int(to_np(rr)[b]) == r_after and 0 <= r_after < N
    assert ((to_np(eng) >= 0) & (to_np(eng) < N)).all()
    Q = 40
    arrival = rng.uniform(0, 20, (3, Q)).round(1).astype(np.float32)
    arrival[:, [3, 17, 18]] = np.nan
    prefill = rng.integers(1, 4, (3, Q)).astype(np.int32)                 # few lengths: arrival order decides most places
    order = torch.full((3, Q), -5, dtype=torch.int32, device=DEV)
    g.order_queues(t(arrival), t(prefill), t(np.full(3, Q, np.int32)), 20.0, order, theta_age=5.0)
    for b in range(3):
        np.testing.assert_array_equal(to_np(order)[b], oracle.order_queue(arrival[b], prefill[b], 20.0, 5.0))
        assert sorted(to_np(order)[b].tolist()) == list(range(Q))


# ------------------------------------------------------------------------------------------
# shapes outside the five configs: the shape-generic scoring kernel, place_check_kernel<0, H>, place_own_r_kernel
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,E,G,sp,S,table_M,counts", [
    (3, 48, 8, 7, 3, False, "i32"),       # E not a power of two, odd slot count, 8 redundant slots
    (2, 160, 64, 3, 5, True, "f32"),      # two ranks per lane, odd slot count, 32 redundant slots, M table
    (2, 200, 16, 16, 4, True, "i32"),     # the largest slot count, 56 redundant slots
    (1, 30, 4, 8, 2, False, "f32"),       # G below a warp: several candidates per warp
])
def test_eval_placements_and_moves_on_other_shapes(L, E, G, sp, S, table_M, counts):
    from workloads.configs import RouterCfg as WRouterCfg, Workload
    NS = G * sp
    w = Workload(name="other", cfg_id=9, router=WRouterCfg(L=L, H=64, E=E, k=2, S=S), T=64, G=G, slots_per_rank=sp, P=72, steps=1,
                 mode=MODE_WINDOW, ema_decay=0.0, window_len=1, zipf_a=1.2, rho=0.5, len_mu=0.0, len_sigma=0.0)
    rng = np.random.default_rng(E + G)
    A = rng.integers(0, 500, (L, S, E)); B = A.sum(1) * rng.integers(20, 60, (L, E))
    if counts == "f32":
        A_t = torch.from_numpy((A * 0.73).astype(np.float32)).to(DEV); B_t = torch.from_numpy((B * 0.73).astype(np.float32)).to(DEV)
    else:
        A_t = torch.from_numpy(A.astype(np.int32)).to(DEV); B_t = torch.from_numpy(B.astype(np.int32)).to(DEV)
    D = gen.comm_cost_D(w, "seeded", DEV)
    M = gen.mig_cost_M(w, DEV) if table_M else None
    prev = gen.prev_placement(w, to_np(B_t), DEV)
    cfg = g.PlacementCfg(L=L, E=E, G=G, slots_per_rank=sp, S=S, counts_dtype=g.COUNTS_F32 if counts == "f32" else g.COUNTS_I32)
    cands = torch.cat([gen.candidates(w, prev, 36, DEV), gen.candidates_redrawn(w, prev, 36, DEV)]).contiguous()
    cands[5, 0, 3] = E                                        # first id past the range (E is not always a power of two)
    c6 = cands[6, L - 1].clone(); c6[1] = c6[0]; cands[6, L - 1] = c6    # twice on rank 0
    out = torch.empty(72, 5, device=DEV); argmin = torch.zeros(1, dtype=torch.int32, device=DEV)
    ws = ws_tensor(g.eval_placements_workspace_bytes(cfg, 72))
    g.eval_placements(cfg, cands, A_t, B_t, D, prev, out, M=M, M_scalar=0.6, argmin=argmin, workspace=ws)
    ref = oracle.objective_batch(to_np(cands), to_np(prev), to_np(A_t), to_np(B_t), to_np(D), to_np(M), 0.6, **_oracle_kw(cfg))
    assert np.isnan(ref[[5, 6]]).all() and not np.isnan(np.delete(ref, [5, 6], 0)).any()
    o = to_np(out).astype(np.float64)
    _check_objective(o, ref)
    assert o[0, 3] == 0.0 and int(argmin.item()) == int(np.nanargmin(to_np(out)[:, 0]))
    # moves: the whole neighbourhood (the staged kernel where it fits, the per-move kernel otherwise) and a list
    cur = cands[2].contiguous()
    n = L * NS * (NS - 1) // 2
    delta = torch.empty(n, 5, device=DEV); best = torch.empty(L, dtype=torch.int32, device=DEV)
    wsm = ws_tensor(g.eval_moves_workspace_bytes(cfg))
    g.eval_moves(cfg, cur, prev, A_t, B_t, D, delta, M=M, M_scalar=0.6, best_per_layer=best, workspace=wsm)
    allmv = oracle.all_pair_moves(L, NS)
    pick = np.arange(n) if n <= 40000 else np.unique(np.concatenate([np.arange(400), np.arange(n - 400, n), rng.integers(0, n, 6000)]))
    refm = oracle.move_deltas(to_np(cur), to_np(prev), allmv[pick], to_np(A_t), to_np(B_t), to_np(D), to_np(M), 0.6, **_oracle_kw(cfg))
    d = to_np(delta).astype(np.float64)
    _check_deltas(cfg, d[pick], refm, allmv[pick], to_np(cur), to_np(A_t), to_np(B_t), to_np(D), to_np(M), 0.6)
    per = n // L
    for l in range(L):
        assert int(best[l].item()) == l * per + int(np.nanargmin(to_np(delta)[l * per:(l + 1) * per, 0]))


@pytest.mark.parametrize("P,L", [(1, 2), (2, 3), (31, 2), (33, 1), (97, 4), (1000, 5), (2051, 58), (4096, 58)])
def test_place_score_tma_kernel_matches_the_lane_load_kernel_and_the_oracle(P, L):
    """The 9 x 32 x 256 shape, scalar M, GIMBAL_PLACE_TRUSTED: rows delivered by TMA (place_score_tma_kernel, the default) against
    the per-lane-load kernel (GIMBAL_OPT_SCORE_TMA = 0) bit for bit -- odd and ragged P (a copy's second candidate past the end,
    chunks that are not a multiple of a warp pass), one block per layer up to the bench grid -- and against the oracle on a
    sample.  Repeated right after a large memset so that every warp's first passes really wait on their barriers; the ring's
    write-after-read ordering (K4) once failed exactly there -- the last case is the bench's own grid
    (P = 4096 candidates x 58 layers, 290 blocks), launched fifty times."""
    w = scaled(get_workload("v3"), L=L, T=256, P=P)
    r = w.router
    rng = np.random.default_rng(11 + P)
    A = torch.from_numpy(rng.integers(0, 3000, (L, r.S, r.E)).astype(np.int32)).to(DEV)
    B = (A.sum(1) * 3).to(torch.int32)
    cfg = g.PlacementCfg(L=L, E=r.E, G=w.G, slots_per_rank=w.slots_per_rank, S=r.S, flags=g.PLACE_TRUSTED)
    D = gen.comm_cost_D(w, "seeded", DEV)
    prev = gen.prev_placement(w, to_np(B), DEV)
    cands = gen.candidates(w, prev, P, DEV)
    ws = ws_tensor(g.eval_placements_workspace_bytes(cfg, P))
    flush = torch.empty(64 << 20, dtype=torch.uint8, device=DEV)
    outs = {}
    for tma in (0, 1):
        g.set_option(g.OPT_SCORE_TMA, tma)
        for rep in range(1 if tma == 0 else (50 if P == 4096 else 12)):
            out = torch.full((P, 5), -3.0, device=DEV)
            flush.zero_()
            g.eval_placements(cfg, cands, A, B, D, prev, out, M_scalar=0.75, workspace=ws)
            torch.cuda.synchronize()
            if tma in outs:
                assert torch.equal(out, outs[tma]), f"run {rep} differs from run 0"
            outs[tma] = out
    assert torch.equal(outs[0], outs[1])
    pick = np.unique(np.concatenate([[0, P - 1, P // 2], rng.integers(0, P, 12)]))
    ref = oracle.objective_batch(to_np(cands)[pick], to_np(prev), to_np(A), to_np(B), to_np(D), None, 0.75, **_oracle_kw(cfg))
    _check_objective(to_np(outs[1]).astype(np.float64)[pick], ref)
    assert to_np(outs[1])[0, 3] == 0.0


@pytest.mark.parametrize("name,hot", [("qwen3", (60, 71)), ("v3", (124, 136)), ("v3", (0, 256)), ("qwen3", (0, 128))])
def test_router_epilogue_parts_meet_on_exact_ties(name, hot):
    """Two epilogue warps per quadrant split a row's experts; ties with the k-th key that span both halves are resolved by the
    total order (key desc, index asc) across the parts.  W rows of the `hot` experts are identical (the others zero), hidden is
    positive: every token's logits tie exactly on the hot experts, and the k lowest hot indices straddle the part boundary
    (E/2) -- or every expert ties.  Reference: the logits-out path (one thread per row), itself checked against the oracle."""
    w = scaled(get_workload(name), L=2, T=700)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    gen_ = torch.Generator(device=DEV).manual_seed(5)
    hidden = (torch.rand(r.L, w.T, r.H, device=DEV, generator=gen_) + 0.25).to(torch.bfloat16)
    u = (torch.rand(r.H, device=DEV, generator=gen_) * 0.02 + 0.01).to(torch.bfloat16)
    W = torch.zeros(r.L, r.E, r.H, dtype=torch.bfloat16, device=DEV)
    W[:, hot[0]:hot[1]] = u
    off = gen.src_offsets(w, 0, w.T, DEV)
    ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
    st = g.StatsState(cfg, MODE_WINDOW, window_len=1)
    logits = torch.empty(r.L, w.T, r.E, device=DEV)
    ids = torch.empty(r.L, w.T, r.k, dtype=torch.int32, device=DEV)
    g.route_stats(cfg, st, T=w.T, hidden=hidden, w_router=W, src_offsets=off, logits_mode=g.LOGITS_OUT, logits=logits, topk_ids=ids, workspace=ws)
    torch.cuda.synchronize()
    offn = to_np(off)
    for l in range(r.L):
        gl = to_np(logits[l])
        assert (gl[:, hot[0]:hot[1]] == gl[:, hot[0]:hot[0] + 1]).all()                 # exact ties on the hot experts
        rid, _ = oracle.gate(gl, r, None, 1)
        np.testing.assert_array_equal(to_np(ids[l]), rid)
        np.testing.assert_array_equal(to_np(st.A_step[l]), oracle.counts(rid, offn, r.S, r.E))
    if hot[1] - hot[0] < r.E and not r.n_groups > 1:
        assert set(np.unique(to_np(ids)).tolist()) == set(range(hot[0], hot[0] + r.k))   # the k lowest hot indices, across E/2
    for parts in (1, 2):
        g.set_option(g.OPT_EPI_PARTS, parts)
        st2 = g.StatsState(cfg, MODE_WINDOW, window_len=1)
        g.route_stats(cfg, st2, T=w.T, hidden=hidden, w_router=W, src_offsets=off, workspace=ws)
        assert torch.equal(st2.A_step, st.A_step), f"epilogue parts = {parts}"


def test_outputs_stay_inside_their_buffers():
    """compute-sanitizer is closed on this pool, so the new store / copy paths are fenced by hand: every output and the workspace sit
    inside larger buffers filled with a sentinel; after the calls the sentinels are intact and only the asked-for slices changed.
    (1) the small-batch router path that STORES a layer's counts, called on a middle slice of the layers; (2) the TMA scoring
    kernel with an odd P (its copies fetch a second candidate past the end) and a workspace of exactly the advertised size."""
    # (1) layers 1..2 of 4, T = 200 (one tile per layer): A_step of layers 0 and 3 must keep the sentinel
    w = scaled(get_workload("v3"), L=4, T=200)
    r = w.router
    cfg = g.RouterCfg.from_workload(r)
    hidden = gen.hidden_all(w, 0, DEV); W = gen.w_router(w, DEV); slb = gen.src_logit_bias(w, 0, DEV); sb = gen.select_bias(w, DEV)
    off = gen.src_offsets(w, 0, w.T, DEV)
    st = g.StatsState(cfg, MODE_WINDOW, window_len=4)
    st.A_step.fill_(-77)
    need = g.route_stats_workspace_bytes(cfg, 2, w.T)
    wsb = torch.full((need + 8192,), 0x5A, dtype=torch.uint8, device=DEV)
    ws = wsb[4096:4096 + need]
    g.route_stats(cfg, st, T=w.T, hidden=hidden[1:3], w_router=W, select_bias=sb, src_logit_bias=slb, src_offsets=off, layer0=1, n_layers=2,
                  workspace=ws)
    torch.cuda.synchronize()
    A = to_np(st.A_step)
    assert (A[0] == -77).all() and (A[3] == -77).all() and (A[1:3] >= 0).all()
    assert A[1:3].sum() == 2 * w.T * r.k and int(st.step_counter.item()) == 0          # not the last slice: no update yet
    assert bool((wsb[:4096] == 0x5A).all()) and bool((wsb[4096 + need:] == 0x5A).all())
    # (2) TMA scoring kernel, P = 37 and 1001
    for P in (37, 1001):
        wp = scaled(get_workload("v3"), L=3, T=256, P=P)
        rng = np.random.default_rng(P)
        A_t = torch.from_numpy(rng.integers(0, 999, (3, r.S, r.E)).astype(np.int32)).to(DEV)
        B_t = A_t.sum(1).to(torch.int32)
        pc = g.PlacementCfg(L=3, E=r.E, G=wp.G, slots_per_rank=wp.slots_per_rank, S=r.S, flags=g.PLACE_TRUSTED)
        D = gen.comm_cost_D(wp, "binary", DEV)
        prev = gen.prev_placement(wp, to_np(B_t), DEV)
        need = g.eval_placements_workspace_bytes(pc, P)
        wsb = torch.full((need + 8192,), 0x5A, dtype=torch.uint8, device=DEV)
        outb = torch.full((P + 64, 5), -5.0, device=DEV)
        candb = torch.zeros(P + 8, 3, wp.NS, dtype=torch.int16, device=DEV)
        candb[:P] = gen.candidates(wp, prev, P, DEV)
        candb[P:] = 255                                                                  # rows past the end: valid ids, never scored
        g.eval_placements(pc, candb[:P], A_t, B_t, D, prev, outb[32:32 + P], workspace=wsb[4096:4096 + need])
        torch.cuda.synchronize()
        assert bool((outb[:32] == -5.0).all()) and bool((outb[32 + P:] == -5.0).all()) and not bool(torch.isnan(outb[32:32 + P]).any())
        assert bool((wsb[:4096] == 0x5A).all()) and bool((wsb[4096 + need:] == 0x5A).all())
        ref = oracle.objective_batch(to_np(candb[:P])[:8], to_np(prev), to_np(A_t), to_np(B_t), to_np(D), None, 1.0, **_oracle_kw(pc))
        _check_objective(to_np(outb[32:40]).astype(np.float64), ref)
