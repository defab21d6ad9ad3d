"""Seeded input generators (torch tensors on the requested device).

Every generator derives its seed from (config id, tag, step, layer) with splitmix64, so
a given (workload, step, layer) always yields the same bytes on a given device type.
Inputs are materialised ONCE per test / bench run and the same bytes are handed to the
CUDA path and to the CPU oracle (copied to host); nothing here is recomputed by either
side.  None of the method's arithmetic lives here: this file draws random numbers,
permutations and request lengths, and applies the skew *recipe* of DESIGN.md section 4.
"""
from __future__ import annotations

import math

import numpy as np
import torch

from .configs import Workload

_MASK = (1 << 64) - 1
_BASE = 0x260615177

TAG_HIDDEN, TAG_W, TAG_RANK_L, TAG_RANK_LS, TAG_SELBIAS, TAG_LEN, TAG_SPIKE, TAG_D, TAG_M, \
    TAG_PREV, TAG_CAND, TAG_MOVES, TAG_DRIFT, TAG_MISC = range(1, 15)


def splitmix64(x: int) -> int:
    x = (x + 0x9E3779B97F4A7C15) & _MASK
    z = x
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
    return z ^ (z >> 31)


def seed_for(cfg_id: int, tag: int, step: int = 0, layer: int = 0) -> int:
    return splitmix64(_BASE ^ (cfg_id << 48) ^ (tag << 40) ^ ((step & 0xFFFFFF) << 16) ^ (layer & 0xFFFF)) & ((1 << 63) - 1)


def _tgen(device, seed: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def _nrng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


# --------------------------------------------------------------------------------------
# router side
# --------------------------------------------------------------------------------------
def hidden_layer(w: Workload, step: int, layer: int, device="cpu", out: torch.Tensor | None = None,
                 T: int | None = None) -> torch.Tensor:
    """hidden[l] ~ N(0,1) -> bf16, [T,H]; distinct per (step, layer)."""
    T = w.T if T is None else T
    H = w.router.H
    g = _tgen(device, seed_for(w.cfg_id, TAG_HIDDEN, step, layer))
    if out is None:
        out = torch.empty(T, H, dtype=torch.bfloat16, device=device)
    # chunked so the fp32 temporary stays small next to the bf16 result
    rows = max(1, (64 << 20) // (4 * H))
    for r0 in range(0, T, rows):
        r1 = min(T, r0 + rows)
        out[r0:r1] = torch.randn(r1 - r0, H, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
    return out


def hidden_all(w: Workload, step: int, device="cpu", layers=None, T: int | None = None) -> torch.Tensor:
    """[n_layers,T,H] bf16 for the given layers (default: all)."""
    layers = list(range(w.router.L)) if layers is None else list(layers)
    T = w.T if T is None else T
    out = torch.empty(len(layers), T, w.router.H, dtype=torch.bfloat16, device=device)
    for i, l in enumerate(layers):
        hidden_layer(w, step, l, device, out=out[i], T=T)
    return out


def w_router(w: Workload, device="cpu") -> torch.Tensor:
    """W_router ~ N(0, 0.02^2) -> bf16, [L,E,H] (row e of layer l is expert e's weight)."""
    r = w.router
    out = torch.empty(r.L, r.E, r.H, dtype=torch.bfloat16, device=device)
    for l in range(r.L):
        g = _tgen(device, seed_for(w.cfg_id, TAG_W, 0, l))
        out[l] = (0.02 * torch.randn(r.E, r.H, generator=g, device=device, dtype=torch.float32)).to(torch.bfloat16)
    return out


def _ranks(w: Workload, step: int):
    """Seeded popularity ranks: rank_l [L,E] and rank_ls [L,S,E], values 1..E, with the
    V3 config's drift (E/16 random rank pairs exchanged every `drift_every` steps)."""
    r = w.router
    rank_l = np.empty((r.L, r.E), dtype=np.int64)
    rank_ls = np.empty((r.L, r.S, r.E), dtype=np.int64)
    for l in range(r.L):
        rank_l[l] = _nrng(seed_for(w.cfg_id, TAG_RANK_L, 0, l)).permutation(r.E) + 1
        rg = _nrng(seed_for(w.cfg_id, TAG_RANK_LS, 0, l))
        for s in range(r.S):
            rank_ls[l, s] = rg.permutation(r.E) + 1
    if w.drift_every > 0:
        for epoch in range(1, step // w.drift_every + 1):
            rg = _nrng(seed_for(w.cfg_id, TAG_DRIFT, epoch, 0))
            for l in range(r.L):
                for _ in range(max(1, r.E // 16)):
                    a, b = rg.choice(r.E, size=2, replace=False)
                    rank_l[l, [a, b]] = rank_l[l, [b, a]]
    return rank_l, rank_ls


def src_logit_bias(w: Workload, step: int = 0, device="cpu") -> torch.Tensor:
    """Benchmark scaffolding that injects the expert skew (not a paper quantity):
    bias[l,s,e] = -a * ( rho*ln rank_l(e) + (1-rho)*ln rank_ls(e) ), fp32 [L,S,E]."""
    rank_l, rank_ls = _ranks(w, step)
    b = -w.zipf_a * (w.rho * np.log(rank_l)[:, None, :] + (1.0 - w.rho) * np.log(rank_ls))
    return torch.from_numpy(b.astype(np.float32)).to(device)


def select_bias(w: Workload, device="cpu") -> torch.Tensor | None:
    """Per-expert selection bias ~ N(0, std^2), fp32 [L,E] (sigmoid configs only)."""
    if w.select_bias_std <= 0.0:
        return None
    r = w.router
    rg = _nrng(seed_for(w.cfg_id, TAG_SELBIAS))
    return torch.from_numpy((w.select_bias_std * rg.standard_normal((r.L, r.E))).astype(np.float32)).to(device)


def src_offsets(w: Workload, step: int = 0, T: int | None = None, device="cpu") -> torch.Tensor:
    """Tokens of a step are concatenated by source DP engine: int32 [S+1]."""
    T = w.T if T is None else T
    S = w.router.S
    counts = np.zeros(S, dtype=np.int64)
    if w.len_mu <= 0.0:
        if S == 2:                       # tiny: 60/40
            counts[0] = int(round(0.6 * T))
            counts[1] = T - counts[0]
        else:                            # decode: equal split
            counts[:] = T // S
            counts[: T % S] += 1
    else:
        rg = _nrng(seed_for(w.cfg_id, TAG_LEN, step))
        mult = np.ones(S, dtype=np.int64)
        if w.bursty:                     # rate x4 with probability 0.1 per source and step
            spikes = _nrng(seed_for(w.cfg_id, TAG_SPIKE, step)).random(S) < 0.1
            mult[spikes] = 4
        order = np.repeat(np.arange(S), mult)    # round-robin dispatch
        left, i = T, 0
        while left > 0:
            n = int(math.ceil(rg.lognormal(w.len_mu, w.len_sigma)))
            n = min(max(n, 1), left)
            counts[order[i % len(order)]] += n
            left -= n
            i += 1
    off = np.zeros(S + 1, dtype=np.int32)
    off[1:] = np.cumsum(counts)
    assert off[-1] == T
    return torch.from_numpy(off).to(device)


# --------------------------------------------------------------------------------------
# placement side
# --------------------------------------------------------------------------------------
def dp_of_rank(w: Workload, device="cpu") -> torch.Tensor:
    """Rank ownership: each DP group's GPUs are its EP ranks: int32 [G]."""
    g = np.arange(w.G, dtype=np.int64)
    return torch.from_numpy((g * w.router.S // w.G).astype(np.int32)).to(device)


def comm_cost_D(w: Workload, kind: str = "binary", device="cpu") -> torch.Tensor:
    """D[s,g] (PAPER.md:242 gives no values): 'binary' = 0 on the source's own DP group, 1
    elsewhere (then C_comm counts remote tokens, Fig. 4); 'seeded' = non-uniform costs."""
    S, G = w.router.S, w.G
    own = (np.arange(G)[None, :] * S // G) == np.arange(S)[:, None]
    if kind == "binary":
        D = np.where(own, 0.0, 1.0)
    else:
        rg = _nrng(seed_for(w.cfg_id, TAG_D))
        D = np.where(own, 0.0, 1.0 + rg.random((S, G)))
    return torch.from_numpy(D.astype(np.float32)).to(device)


def mig_cost_M(w: Workload, device="cpu") -> torch.Tensor:
    """Seeded M[l,e,g] = 1 + 0.5*U(0,1), fp32 [L,E,G] (PAPER.md:250 gives no values)."""
    r = w.router
    rg = _nrng(seed_for(w.cfg_id, TAG_M))
    return torch.from_numpy((1.0 + 0.5 * rg.random((r.L, r.E, w.G))).astype(np.float32)).to(device)


def _colocated(rows: torch.Tensor, G: int, sp: int) -> torch.Tensor:
    """[N,G] bool: rank holds the same expert twice."""
    x = rows.view(rows.shape[0], G, sp).to(torch.int32)
    s, _ = torch.sort(x, dim=-1)
    return (s[..., 1:] == s[..., :-1]).any(-1)


def _repair(rows: torch.Tensor, G: int, sp: int, gen: torch.Generator) -> torch.Tensor:
    """Random slot exchanges until no rank holds two copies of one expert (x stays binary)."""
    N, NS = rows.shape
    dev = rows.device
    for _ in range(200):
        dup = _colocated(rows, G, sp)
        bad = dup.any(-1).nonzero().flatten()
        if bad.numel() == 0:
            return rows
        g = dup[bad].to(torch.int8).argmax(-1)                       # first bad rank
        seg = rows[bad].view(-1, G, sp)[torch.arange(bad.numel(), device=dev), g].to(torch.int32)
        eq = (seg[:, :, None] == seg[:, None, :]) & torch.tril(torch.ones(sp, sp, dtype=torch.bool, device=dev), -1)
        j = eq.any(-1).to(torch.int8).argmax(-1)                     # a later copy inside that rank
        a = g * sp + j
        b = torch.randint(0, NS, (bad.numel(),), generator=gen, device=dev)
        va, vb = rows[bad, a].clone(), rows[bad, b].clone()
        rows[bad, a], rows[bad, b] = vb, va
    raise RuntimeError("placement repair did not converge")


def prev_placement(w: Workload, B, device="cpu") -> torch.Tensor:
    """x0: a seeded random valid placement per layer, int16 [L,NS] slot -> expert; the
    NS-E redundant slots replicate the highest-B experts of that layer (B: [L,E] array)."""
    r = w.router
    NS, E = w.NS, r.E
    Bn = np.asarray(B, dtype=np.float64).reshape(r.L, E)
    rows = np.empty((r.L, NS), dtype=np.int16)
    for l in range(r.L):
        extra = np.argsort(-Bn[l], kind="stable")[np.arange(NS - E) % E]
        base = np.concatenate([np.arange(E), extra]).astype(np.int16)
        rows[l] = _nrng(seed_for(w.cfg_id, TAG_PREV, 0, l)).permutation(base)
    t = torch.from_numpy(rows).to(device)
    return _repair(t, w.G, w.slots_per_rank, _tgen(device, seed_for(w.cfg_id, TAG_PREV, 1)))


def candidates(w: Workload, prev: torch.Tensor, P: int | None = None, device="cpu") -> torch.Tensor:
    """[P,L,NS] int16.  p=0 is x0 itself; the first half are x0 with 1..16 random slot
    transpositions per layer; the second half are random permutations of the slot contents."""
    P = w.P if P is None else P
    L, NS = prev.shape
    prev = prev.to(device)
    gen = _tgen(device, seed_for(w.cfg_id, TAG_CAND))
    out = prev.unsqueeze(0).repeat(P, 1, 1).contiguous()
    half = max(1, P // 2)
    if half > 1:
        near = out[1:half].reshape(-1, NS)
        N = near.shape[0]
        n_sw = torch.randint(1, 17, (N,), generator=gen, device=device)
        ar = torch.arange(N, device=device)
        for t in range(16):
            a = torch.randint(0, NS, (N,), generator=gen, device=device)
            b = torch.randint(0, NS, (N,), generator=gen, device=device)
            act = n_sw > t
            va, vb = near[ar, a].clone(), near[ar, b].clone()
            near[ar, a] = torch.where(act, vb, va)
            near[ar, b] = torch.where(act, va, near[ar, b])
        out[1:half] = _repair(near, w.G, w.slots_per_rank, gen).view(half - 1, L, NS)
    if P > half:
        far = out[half:].reshape(-1, NS)
        chunk = max(1, (32 << 20) // NS)
        for r0 in range(0, far.shape[0], chunk):
            blk = far[r0:r0 + chunk]
            perm = torch.rand(blk.shape, generator=gen, device=device).argsort(-1)
            far[r0:r0 + chunk] = torch.gather(blk, 1, perm)
        out[half:] = _repair(far, w.G, w.slots_per_rank, gen).view(P - half, L, NS)
    return out


def candidates_redrawn(w: Workload, prev: torch.Tensor, P: int | None = None, device="cpu") -> torch.Tensor:
    """[P,L,NS] int16 like `candidates`, but every (candidate, layer) draws its own NS - E redundant copies
    (uniformly, with repetition: an expert may get 3 or more ranks), so the replica counts differ from x0's --
    what a rebalancer searches over when it decides WHICH hot experts to replicate (EPLB-style).
    p=0 stays x0.  Without redundant slots (NS == E) this is a random permutation."""
    P = w.P if P is None else P
    L, NS = prev.shape
    E = w.router.E
    prev = prev.to(device)
    gen = _tgen(device, seed_for(w.cfg_id, TAG_CAND, 1))
    base = torch.arange(E, device=device, dtype=torch.int16).repeat(P * L, 1)
    if NS > E:
        extra = torch.randint(0, E, (P * L, NS - E), generator=gen, device=device).to(torch.int16)
        base = torch.cat([base, extra], dim=1)
    perm = torch.rand(base.shape, generator=gen, device=device).argsort(-1)
    rows = _repair(torch.gather(base, 1, perm), w.G, w.slots_per_rank, gen)
    out = rows.view(P, L, NS).contiguous()
    out[0] = prev
    return out


def to_expert_rank_u8(cands: torch.Tensor, sp: int) -> torch.Tensor:
    """slot -> expert rows [..., NS] (no replicas, NS == E) -> expert -> rank bytes [..., E] (the EXPERT_TO_RANK_U8
    candidate encoding of include/gimbal.h).  Pure re-indexing."""
    NS = cands.shape[-1]
    flat = cands.reshape(-1, NS).long()
    rank = (torch.arange(NS, device=cands.device) // sp).to(torch.uint8).expand_as(flat)
    out = torch.empty_like(flat, dtype=torch.uint8)
    out.scatter_(1, flat, rank)
    return out.view(*cands.shape[:-1], NS).contiguous()


def explicit_moves(w: Workload, n: int, device="cpu") -> torch.Tensor:
    """[n,3] int32 (layer, slot_a, slot_b), slot_a != slot_b."""
    gen = _tgen(device, seed_for(w.cfg_id, TAG_MOVES))
    l = torch.randint(0, w.router.L, (n,), generator=gen, device=device)
    a = torch.randint(0, w.NS, (n,), generator=gen, device=device)
    d = torch.randint(1, w.NS, (n,), generator=gen, device=device)
    b = (a + d) % w.NS
    return torch.stack([l, a, b], dim=1).to(torch.int32)
