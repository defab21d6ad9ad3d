"""gimbal_route_stats_static: the routing-statistics step for callers that cannot allocate device memory.

Some users of this library have no workspace to hand over and no way to get one: a scheduler thread inside a
serving engine whose HBM went to the KV-cache pool at start-up (a later cudaMalloc fails or eats into that
pool), or a side thread for which the device-wide stall of cudaMalloc / cudaFree next to a running decode loop
is not acceptable.  For them the scratch of the a4-a5 update (pressure partials + the layer counter) is a
64 KiB `static __device__` array inside libgimbal.so -- one per GPU, shared by every call, never cleared
behind the caller's back except when the shape's scratch layout changes.

What is checked here: on the same seeded inputs, two steps in a row through the new entry point leave
exactly what the workspace path leaves -- ids, counts, window / EMA profile, B, pressure, step counter --
for a sequence of shapes chosen so that each one finds the previous shape's leftovers in the array
(throughput regime, small-batch regime with the update fused into the router kernel, gating on given
logits, layer-sliced calls).  Integers are compared bit for bit; floats to the 1e-5 the other tests use
(they are in fact identical: same kernels, same launch configuration).  The size limit is checked too.

The file is named to be collected last (`pytest --collect-only`): under `pytest -x` a failure here hides
nothing behind it.  It passes alone in a fresh process (array still zero from load) and after the rest of
the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_2606_15177_b200 as g
from tests.util import ws_tensor
from workloads import gen, get_workload, scaled
from workloads.configs import MODE_EMA, MODE_WINDOW

DEV = "cuda"

# (workload, L, T, profile mode, how the step is issued) -- in this order: every shape after the first finds
# leftovers in the array (v3 with L = 6 writes 768 bytes of partials and keeps its layer counter behind them; the
# shapes that follow have at most 256 bytes of partials and their counter at byte 256, inside v3's partials)
SEQUENCE = [
    ("v3", 6, 1100, MODE_WINDOW, "fused"),
    ("tiny", 1, 1000, MODE_EMA, "fused"),
    ("v2lite", 3, 1500, MODE_EMA, "logits_in"),
    ("decode", 2, 256, MODE_EMA, "fused"),         # small-batch regime: update inside the router kernel
    ("qwen3", 2, 1300, MODE_WINDOW, "sliced"),
]


def _same(a, b, what):
    if a.dtype.is_floating_point:
        torch.testing.assert_close(a, b, rtol=1e-5, atol=0.0, msg=lambda m: f"{what}: {m}")
    else:
        assert torch.equal(a, b), what


def _issue(fn, how, cfg, st, w, inputs, ids, extra):
    hidden, W, slb, sb, off, logits = inputs
    r = w.router
    kw = dict(T=w.T, select_bias=sb, src_offsets=off, cur_placement=extra["place"], dp_of_rank=extra["dp"], G=w.G,
              slots_per_rank=w.slots_per_rank, **extra["ws"])
    if how == "logits_in":
        fn(cfg, st, logits_mode=g.LOGITS_IN, logits=logits, topk_ids=ids, **kw)
    elif how == "sliced":
        for l in range(r.L):
            fn(cfg, st, hidden=hidden[l:l + 1], w_router=W, src_logit_bias=slb, layer0=l, n_layers=1, topk_ids=ids[l:l + 1], **kw)
    else:
        fn(cfg, st, hidden=hidden, w_router=W, src_logit_bias=slb, topk_ids=ids, **kw)


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_workspace_path_on_two_calls_in_a_row():
    for name, L, T, mode, how in SEQUENCE:
        w = scaled(get_workload(name), L=L, T=T, P=16)
        r = w.router
        cfg = g.RouterCfg.from_workload(r)
        place = gen.prev_placement(w, np.random.default_rng(5).integers(1, 1000, (r.L, r.E)), DEV)
        dp = gen.dp_of_rank(w, DEV)
        W, sb = gen.w_router(w, DEV), gen.select_bias(w, DEV)
        ws = ws_tensor(g.route_stats_workspace_bytes(cfg, r.L, w.T))
        assert g.route_stats_workspace_bytes(cfg, r.L, w.T) <= g.STATIC_SCRATCH_BYTES
        st_ws = g.StatsState(cfg, mode, window_len=2, ema_decay=0.9)
        st_static = g.StatsState(cfg, mode, window_len=2, ema_decay=0.9)
        for step in range(2):                                   # two calls in a row, the second on the first one's leftovers
            hidden = gen.hidden_all(w, step, DEV)
            slb = gen.src_logit_bias(w, step, DEV)
            off = gen.src_offsets(w, step, w.T, DEV)
            logits = None
            if how == "logits_in":
                gen_ = torch.Generator(device=DEV); gen_.manual_seed(40 + step)
                logits = (torch.randn(r.L, w.T, r.E, generator=gen_, device=DEV) * 1.7).contiguous()
            inputs = (hidden, W, slb, sb, off, logits)
            ids_ws = torch.full((r.L, w.T, r.k), -9, dtype=torch.int32, device=DEV)
            ids_static = torch.full_like(ids_ws, -7)
            _issue(g.route_stats, how, cfg, st_ws, w, inputs, ids_ws, dict(place=place, dp=dp, ws=dict(workspace=ws)))
            _issue(g.route_stats_static, how, cfg, st_static, w, inputs, ids_static, dict(place=place, dp=dp, ws={}))
            torch.cuda.synchronize()
            tag = f"{name} / {how} / step {step}"
            _same(ids_static, ids_ws, f"{tag}: top-k ids")
            for field in ("A_step", "A_win", "A_pub", "B_pub", "A_ema", "B", "pressure_raw", "pressure_rel", "step_counter", "status"):
                _same(getattr(st_static, field), getattr(st_ws, field), f"{tag}: {field}")
            assert int(st_static.step_counter.item()) == step + 1 and int(st_static.status.item()) == 0, tag
            assert int(st_static.A_step.sum().item()) == r.L * w.T * r.k, tag          # every routed token was counted
            assert float(st_static.pressure_raw.sum().item()) > 0.0, tag               # and the pressure came out of the array


def test_static_scratch_entry_point_refuses_shapes_beyond_its_array():
    """L * S = 8192 needs 66,048 bytes of scratch: refused on the host with both sizes in the message, before any
    device is touched (so this runs on a CPU box too); the largest shape that fits passes this check."""
    st = g.binding._StatsState()
    too_big = g.RouterCfg(L=128, H=256, E=64, k=2, S=64)
    c = too_big.c()
    assert g.route_stats_workspace_bytes(too_big, 128, 16) > g.STATIC_SCRATCH_BYTES
    rc = g.lib().gimbal_route_stats_static(C.byref(c), 0, 128, 16, None, None, None, None, None, 0, None, None, None, None, None, 0, 0,
                                           C.byref(st), None, None)
    msg = g.last_error()
    assert rc == -4 and "66048" in msg and "65536" in msg and "workspace of your own" in msg
    fits = g.RouterCfg(L=127, H=256, E=64, k=2, S=64)          # 8128 partials: exactly the array
    c = fits.c()
    assert g.route_stats_workspace_bytes(fits, 127, 16) == g.STATIC_SCRATCH_BYTES
    rc = g.lib().gimbal_route_stats_static(C.byref(c), 0, 127, 16, None, None, None, None, None, 0, None, None, None, None, None, 0, 0,
                                           C.byref(st), None, None)
    assert rc != -4                                            # goes on to the device probe / argument checks instead
