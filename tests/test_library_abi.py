"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol that
include/gimbal.h declares, validates arguments on the host, and refuses to compute without a
GPU (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest
import torch

import paper_2606_15177_b200 as g

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "gimbal.h")).read()
    return sorted(set(re.findall(r"GIMBAL_API\s+[\w\s\*]+?\b(gimbal_\w+)\s*\(", src)))


def test_build_is_current_and_loads():
    from paper_2606_15177_b200 import build
    build.build()
    assert g.lib().gimbal_version() == g.ABI_VERSION == 300


def test_every_declared_symbol_is_exported():
    decl = _declared_symbols()
    assert len(decl) >= 12
    assert sorted(decl) == sorted(g.EXPORTED_SYMBOLS)
    for name in decl:
        assert hasattr(g.lib(), name), name


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_15177_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "gimbal_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_15177_b200" not in txt and "from paper_2606_15177_b200" not in txt and "csrc" not in txt.replace("under paper_2606_15177_b200/csrc", ""), f


def test_host_side_validation():
    cfg = g.RouterCfg(L=2, H=256, E=48, k=2, S=2)            # E not supported
    c = cfg.c()
    st = g.binding._StatsState()
    rc = g.lib().gimbal_route_stats(C.byref(c), 0, 2, 16, None, None, None, None, None, 0, None, None, None, None, None, 0, 0,
                                    C.byref(st), None, None, C.c_size_t(0), None)
    assert rc == -2 and "E=48" in g.last_error()
    cfg = g.RouterCfg(L=2, H=250, E=64, k=2, S=2)
    c = cfg.c()
    rc = g.lib().gimbal_route_stats(C.byref(c), 0, 2, 16, None, None, None, None, None, 0, None, None, None, None, None, 0, 0,
                                    C.byref(st), None, None, C.c_size_t(0), None)
    assert rc == -2 and "multiple of 64" in g.last_error()
    cfg = g.RouterCfg(L=2, H=256, E=64, k=2, S=2)
    c = cfg.c()
    rc = g.lib().gimbal_route_stats(C.byref(c), 0, 3, 16, None, None, None, None, None, 0, None, None, None, None, None, 0, 0,
                                    C.byref(st), None, None, C.c_size_t(0), None)
    assert rc == -1 and "layer range" in g.last_error()
    pc = g.PlacementCfg(L=1, E=16, G=3, slots_per_rank=6, S=2).c()
    rc = g.lib().gimbal_eval_placements(C.byref(pc), 1, None, None, None, None, None, C.c_float(1.0), None, None, None, None,
                                        C.c_size_t(0), None)
    assert rc == -2 and "power of two" in g.last_error()
    # one rank with an odd number of slots: rows of odd length would be read through misaligned 32-bit words
    pc = g.PlacementCfg(L=2, E=2, G=1, slots_per_rank=3, S=2).c()
    rc = g.lib().gimbal_eval_placements(C.byref(pc), 1, None, None, None, None, None, C.c_float(1.0), None, None, None, None,
                                        C.c_size_t(0), None)
    assert rc == -2 and "must be even" in g.last_error()
    assert g.eval_placements_workspace_bytes(g.PlacementCfg(L=58, E=256, G=32, slots_per_rank=9, S=16), 4096) > 58 * 256 * 32 * 8


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback_without_gpu():
    cfg = g.RouterCfg(L=1, H=256, E=16, k=2, S=2)
    c = cfg.c()
    st = g.binding._StatsState()
    one = C.c_void_p(16)          # fake non-NULL, 16-byte aligned "device" pointers: never dereferenced on the host
    st.A_step = st.A_win = st.A_pub = st.B_pub = st.B = st.step_counter = 16
    st.mode, st.window_len, st.abi_version = 0, 1, g.ABI_VERSION
    rc = g.lib().gimbal_route_stats(C.byref(c), 0, 1, 16, one, one, None, None, one, 0, None, None, None, None, None, 0, 0,
                                    C.byref(st), None, one, C.c_size_t(1 << 20), None)
    assert rc == -2 and "CUDA" in g.last_error()


def test_options_are_validated_and_readable():
    """gimbal_set_option / gimbal_get_option: defaults, ranges (nothing reads the environment)."""
    defaults = {g.OPT_CTA_GROUP: 0, g.OPT_FUSE_GATE: 1, g.OPT_SCORE_GENERIC: 0, g.OPT_CHECK_SCORES_ALL: 0, g.OPT_HIST_AGG: 1,
                g.OPT_SCORE_TMA: 1, g.OPT_EPI_PARTS: 0, g.OPT_PDL: 1, g.OPT_FUSE_UPDATE: 1}
    for opt, val in defaults.items():
        assert g.get_option(opt) == val
    for opt in (g.OPT_CTA_GROUP, g.OPT_EPI_PARTS, g.OPT_PDL):
        assert g.lib().gimbal_set_option(opt, 3) == -1 and g.lib().gimbal_set_option(opt, 2) == 0 and g.get_option(opt) == 2
        g.set_option(opt, defaults[opt])
    for opt in (g.OPT_SCORE_TMA, g.OPT_HIST_AGG, g.OPT_FUSE_UPDATE):
        assert g.lib().gimbal_set_option(opt, 2) == -1 and g.get_option(opt) == 1
    assert g.lib().gimbal_set_option(99, 0) == -1


def test_structs_laid_out_by_another_header_are_refused():
    """A caller compiled against the round-1 header passes a state whose step_counter is i64[1] and whose `reserved` word is 0,
    and a placement cfg that ends before `encoding` / `flags` (whatever follows it in memory is read there): both are refused on
    the host, before anything is launched, instead of being written or read out of bounds."""
    cfg = g.RouterCfg(L=1, H=256, E=16, k=2, S=2)
    c = cfg.c()
    st = g.binding._StatsState()
    one = C.c_void_p(16)
    st.A_step = st.A_win = st.A_pub = st.B_pub = st.B = st.step_counter = 16
    st.mode, st.window_len = 0, 1                                   # abi_version left at 0, as `reserved` was
    rc = g.lib().gimbal_route_stats(C.byref(c), 0, 1, 16, one, one, None, None, one, 0, None, None, None, None, None, 0, 0,
                                    C.byref(st), None, one, C.c_size_t(1 << 20), None)
    assert rc == -1 and "abi_version=0" in g.last_error() and "300" in g.last_error()
    rc = g.lib().gimbal_route_stats_static(C.byref(c), 0, 1, 16, one, one, None, None, one, 0, None, None, None, None, None, 0, 0,
                                           C.byref(st), None, None)
    assert rc in (-1, -2)                                          # -2 on a CPU box (the device probe comes first on this entry point)
    for enc, flags, what in ((2, 0, "encoding=2"), (0, 6, "flags=0x6"), (-1, 0, "encoding=-1")):
        pc = g.PlacementCfg(L=1, E=16, G=4, slots_per_rank=4, S=2, encoding=enc, flags=flags).c()
        rc = g.lib().gimbal_eval_placements(C.byref(pc), 1, None, None, None, None, None, C.c_float(1.0), None, None, None, None,
                                            C.c_size_t(0), None)
        assert rc == -1 and what in g.last_error()
        assert g.lib().gimbal_eval_moves(C.byref(pc), None, None, C.c_int64(0), None, None, None, None, None, C.c_float(1.0), None, None,
                                         None, C.c_size_t(0), None) == -1
