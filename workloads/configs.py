"""Shapes of the five BASELINE.json configs (SURVEY.md section 8, table "Config shapes").

Pure data: no arithmetic of the method lives here.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

SOFTMAX = 0
SIGMOID = 1

MODE_WINDOW = 0
MODE_EMA = 1


@dataclass(frozen=True)
class RouterCfg:
    """Router / gating shape.  Gating math is fixed by BASELINE.json's model-shaped
    configs, the paper only says "top-k"; reading R1."""
    L: int            # MoE layers
    H: int            # hidden size
    E: int            # logical (routed) experts
    k: int            # top-k
    S: int            # source DP engines
    score_fn: int = SOFTMAX
    renorm: int = 0
    n_groups: int = 1
    topk_groups: int = 1
    group_score_topn: int = 1
    routed_scale: float = 1.0


@dataclass(frozen=True)
class Workload:
    name: str
    cfg_id: int               # index in BASELINE.json.configs (seed derivation)
    router: RouterCfg
    T: int                    # tokens per step
    G: int                    # logical EP ranks
    slots_per_rank: int
    P: int                    # candidate placements per scoring call
    steps: int                # steps of the stats path in one "episode"
    mode: int                 # MODE_WINDOW / MODE_EMA
    ema_decay: float
    window_len: int
    zipf_a: float             # expert-skew exponent
    rho: float                # 1 = source independent skew, <1 = source dependent
    len_mu: float             # lognormal prompt-length parameters (0 = fixed split)
    len_sigma: float
    bursty: bool = False      # Poisson-driven per-source rate spikes (Qwen3 config)
    drift_every: int = 0      # skew drifts every N steps (V3 config)
    select_bias_std: float = 0.0
    rescore_every: int = 0    # decode config: placement re-score period

    @property
    def NS(self) -> int:
        return self.G * self.slots_per_rank


WORKLOADS = {
    # tiny: 1 layer, hidden 256, 16 experts, top-2 softmax, 2 sources, 4096 tokens 60/40;
    # 16 experts onto 4 ranks x 4 slots, 64 candidates + all 120 swaps.
    "tiny": Workload(
        name="tiny", cfg_id=0,
        router=RouterCfg(L=1, H=256, E=16, k=2, S=2),
        T=4096, G=4, slots_per_rank=4, P=64, steps=1, mode=MODE_WINDOW, ema_decay=0.0,
        window_len=1, zipf_a=1.1, rho=1.0, len_mu=0.0, len_sigma=0.0),
    # DeepSeek-V2-Lite-shaped: 26 layers, hidden 2048, 64 experts, top-6 softmax, 4 sources,
    # 16384 tokens, EMA 0.9 over 32 steps; 8 ranks x 8 slots, 1024 candidates.
    "v2lite": Workload(
        name="v2lite", cfg_id=1,
        router=RouterCfg(L=26, H=2048, E=64, k=6, S=4),
        T=16384, G=8, slots_per_rank=8, P=1024, steps=32, mode=MODE_EMA, ema_decay=0.9,
        window_len=32, zipf_a=1.2, rho=0.5, len_mu=6.0, len_sigma=1.0),
    # Qwen3-30B-A3B-shaped: 48 layers, hidden 2048, 128 experts, top-8 softmax + renorm,
    # 8 sources, 32768 tokens, bursty arrivals; 16 ranks x 8 slots, 2048 candidates.
    "qwen3": Workload(
        name="qwen3", cfg_id=2,
        router=RouterCfg(L=48, H=2048, E=128, k=8, S=8, renorm=1),
        T=32768, G=16, slots_per_rank=8, P=2048, steps=32, mode=MODE_WINDOW, ema_decay=0.0,
        window_len=32, zipf_a=1.2, rho=0.5, len_mu=6.5, len_sigma=1.2, bursty=True),
    # DeepSeek-V3-shaped: 58 layers, hidden 7168, 256 experts, sigmoid + bias, 8 groups /
    # top-4 groups, top-8, 16 sources, 65536 tokens, skew drifting every 8 steps;
    # 288 slots (256 + 32 replicas) on 32 ranks, 4096 candidates + full move neighbourhood.
    "v3": Workload(
        name="v3", cfg_id=3,
        router=RouterCfg(L=58, H=7168, E=256, k=8, S=16, score_fn=SIGMOID, renorm=1,
                         n_groups=8, topk_groups=4, group_score_topn=2, routed_scale=2.5),
        T=65536, G=32, slots_per_rank=9, P=4096, steps=24, mode=MODE_WINDOW, ema_decay=0.0,
        window_len=8, zipf_a=1.3, rho=0.5, len_mu=6.5, len_sigma=1.2, drift_every=8,
        select_bias_std=0.05),
    # decode-streaming stress: V3 router, 256 tokens/step x 2000 steps, EMA update each
    # step, re-score 16384 candidates on 64 ranks every 100 steps.
    "decode": Workload(
        name="decode", cfg_id=4,
        router=RouterCfg(L=58, H=7168, E=256, k=8, S=16, score_fn=SIGMOID, renorm=1,
                         n_groups=8, topk_groups=4, group_score_topn=2, routed_scale=2.5),
        T=256, G=64, slots_per_rank=4, P=16384, steps=2000, mode=MODE_EMA, ema_decay=0.9,
        window_len=100, zipf_a=1.3, rho=0.5, len_mu=0.0, len_sigma=0.0,
        select_bias_std=0.05, rescore_every=100),
}


def get_workload(name: str) -> Workload:
    return WORKLOADS[name]


def scaled(w: Workload, *, L=None, T=None, H=None, P=None, steps=None) -> Workload:
    """Same gating / placement structure at a size the CPU oracle finishes in seconds."""
    r = w.router
    r2 = replace(r, L=L if L is not None else r.L, H=H if H is not None else r.H)
    return replace(w, router=r2, T=T if T is not None else w.T,
                   P=P if P is not None else w.P,
                   steps=steps if steps is not None else w.steps)
