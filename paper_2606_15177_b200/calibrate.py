"""NEXT-4: calibration of the greedy heuristic's weights against an exhaustive reference -- the analogue of the
paper's Fig. 6 ("we fix alpha = 1.0 and calibrate beta and gamma against an offline MINLP reference
computed from the dumped expert-load and source-DP-to-expert matrices ... preserves more than 80% of the MINLP
placement decisions and keeps source-aware communication within 0.6% of the offline reference").

No MINLP solver and none of the paper's dumps are available, so the reference here is the exact minimiser of the
printed objective C_load + C_comm + C_mig found by scoring EVERY placement of a small instance with
gimbal_eval_placements, and the heuristic is gimbal_greedy_place.  Orchestration only: all arithmetic runs in the
library's kernels.
"""
from __future__ import annotations

import itertools

import numpy as np
import torch

from . import binding as g


def all_placements(E: int, G: int, sp: int) -> np.ndarray:
    """Every assignment of E = G*sp experts to G ranks of sp slots, as slot -> expert rows [n, E] (experts of a rank in
    ascending order): E! / (sp!)^G rows, e.g. 2,520 for 8 experts on 4 x 2 slots."""
    assert E == G * sp
    rows = []

    def rec(remaining, acc):
        if not remaining:
            rows.append([e for grp in acc for e in grp])
            return
        for grp in itertools.combinations(remaining, sp):            # the next rank's experts
            rec([e for e in remaining if e not in grp], acc + [grp])

    rec(list(range(E)), [])
    return np.asarray(rows, dtype=np.int16)


def rank_of(placement: np.ndarray, sp: int) -> np.ndarray:
    """slot -> expert row [NS] -> expert -> rank [E] (no replicas)."""
    out = np.empty(placement.shape[-1], dtype=np.int64)
    out[placement.astype(np.int64)] = np.arange(placement.shape[-1]) // sp
    return out


def calibration_sweep(A, B, D, prev, G: int, sp: int, betas, gammas, M_scalar: float = 1.0, device="cuda"):
    """A [n,S,E], B [n,E] integer counts of n independent one-layer instances, D [S,G], prev [n,NS] (x0).
    Returns dict(agree [nb,ng], comm_gap [nb,ng], best=(beta, gamma), ref [n,NS]):
      agree     mean fraction of experts the heuristic puts on the rank the reference chose ("placement
                decisions preserved");
      comm_gap  mean of C_comm(heuristic) / C_comm(reference) - 1.
    The n instances are passed to the library as the n layers of one problem."""
    A = np.ascontiguousarray(A); B = np.ascontiguousarray(B); prev = np.ascontiguousarray(prev, dtype=np.int16)
    n, S, E = A.shape
    NS = G * sp
    assert NS == E, "the exhaustive reference is for instances without replicas"
    t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(device=device, dtype=dt)
    A_t, B_t, D_t, prev_t = t(A, torch.int32), t(B, torch.int32), t(D, torch.float32), t(prev, torch.int16)
    # ---- reference: exact minimiser of the printed objective (weights 1, 1, 1), instance by instance
    cands = all_placements(E, G, sp)
    P = cands.shape[0]
    cfg1 = g.PlacementCfg(L=1, E=E, G=G, slots_per_rank=sp, S=S, alpha=1.0, beta=1.0, gamma=1.0)
    ws = torch.empty(g.eval_placements_workspace_bytes(cfg1, P), dtype=torch.uint8, device=device)
    cand_t = t(cands[:, None, :], torch.int16)
    out = torch.empty(P, 5, device=device)
    argmin = torch.zeros(1, dtype=torch.int32, device=device)
    ref = np.empty((n, NS), dtype=np.int16)
    ref_comm = np.empty(n)
    for i in range(n):
        g.eval_placements(cfg1, cand_t, A_t[i:i + 1], B_t[i:i + 1], D_t, prev_t[i:i + 1], out, M_scalar=M_scalar, argmin=argmin, workspace=ws)
        j = int(argmin.item())
        ref[i] = cands[j]
        ref_comm[i] = float(out[j, 2].item())
    ref_rank = np.stack([rank_of(ref[i], sp) for i in range(n)])
    # ---- the heuristic on every grid point; its communication cost through the same evaluator
    agree = np.empty((len(betas), len(gammas)))
    gap = np.empty_like(agree)
    placed = torch.empty_like(prev_t)
    cfgn = g.PlacementCfg(L=n, E=E, G=G, slots_per_rank=sp, S=S)
    wsn = torch.empty(g.eval_placements_workspace_bytes(cfg1, 1), dtype=torch.uint8, device=device)
    one = torch.empty(1, 5, device=device)
    for bi, beta in enumerate(betas):
        for gi, gamma in enumerate(gammas):
            cfgn.alpha, cfgn.beta, cfgn.gamma = 1.0, float(beta), float(gamma)
            g.greedy_place(cfgn, A_t, B_t, D_t, prev_t, placed, M_scalar=M_scalar)
            got = placed.cpu().numpy()
            same, ratio = [], []
            for i in range(n):
                same.append(float((rank_of(got[i], sp) == ref_rank[i]).mean()))
                g.eval_placements(cfg1, placed[i:i + 1].unsqueeze(0).contiguous(), A_t[i:i + 1], B_t[i:i + 1], D_t, prev_t[i:i + 1], one,
                                  M_scalar=M_scalar, workspace=wsn)
                c = float(one[0, 2].item())
                ratio.append(c / ref_comm[i] - 1.0 if ref_comm[i] > 0 else 0.0)
            agree[bi, gi], gap[bi, gi] = np.mean(same), np.mean(ratio)
    bi, gi = np.unravel_index(np.lexsort((np.abs(gap).ravel(), -agree.ravel()))[0], agree.shape)
    return dict(agree=agree, comm_gap=gap, best=(float(betas[bi]), float(gammas[gi])), ref=ref, ref_comm=ref_comm)
