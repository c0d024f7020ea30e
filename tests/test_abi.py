"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/sk_b200.h declares,
and rejects bad arguments before touching the device (no compute call is made here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sk():
    import paper_1808_10365_b200 as m
    from paper_1808_10365_b200 import build
    build.build()                      # nvcc cross-compiles for sm_100a without a GPU
    m.lib()
    return m


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "sk_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sk_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(sk):
    names = declared_symbols()
    assert set(names) == set(sk.SYMBOLS)
    raw = C.CDLL(sk.LIB_PATH)
    for n in names:
        assert getattr(raw, n) is not None


def test_product_has_no_measurement_or_override_entries(sk):
    """The product boundary carries no measurement kernels and no process-wide knobs ("no
    globals"): those live in libsk_b200_bench.so, which loads and exports what csrc/bench/sk_bench.h declares."""
    names = declared_symbols()
    assert not [n for n in names if n.startswith("sk_debug")]
    raw = C.CDLL(sk.LIB_PATH)
    for gone in ("sk_debug_set_plan", "sk_debug_get_plan", "sk_debug_loop_ceiling", "sk_debug_pipe_rate"):
        assert not hasattr(raw, gone)
    from paper_1808_10365_b200 import benchlib
    text = open(os.path.join(ROOT, "paper_1808_10365_b200", "csrc", "bench", "sk_bench.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(skb_[a-z_0-9]+)\s*\(", text)))
    assert set(declared) == set(benchlib.SYMBOLS)
    braw = C.CDLL(benchlib.LIB_PATH)
    for n in declared:
        assert getattr(braw, n) is not None
    one = C.c_void_p(256)
    L = benchlib.lib()
    assert L.skb_loop_ceiling(0, 12, 0, one, one, None, None) == -2          # argument errors need no device
    assert L.skb_loop_ceiling(1, 12, 10, one, one, None, None) == -5         # the memory-only variant has no loop form
    assert L.skb_stream_workspace_bytes(49152, 1, 2048, 256) == 192 * 8 * 8 + 192 * 4
    assert L.skb_stream_workspace_bytes(49152, 1, 2048, 512) == 0


def test_plan_override_is_per_call(sk):
    """The SK_FRAME_PLAN_* bits act on the call that carries them and leave nothing behind in the library
    (sk_frame_plan is a pure query, so this needs no device)."""
    auto = sk.sk_frame_plan(49152, 1, 2048, 256, flags=0)
    for lanes in (1, 2, 4, 8, 16):
        assert sk.sk_frame_plan(49152, 1, 2048, 256, flags=sk.plan_flags(lanes=lanes))[0] == lanes
        assert sk.sk_frame_plan(49152, 1, 2048, 256, flags=0) == auto
    assert sk.sk_frame_plan(49152, 1, 2048, 256, flags=sk.plan_flags(sk.SK_PLAN_LDG))[2] == 0     # direct-load kernel
    assert sk.sk_frame_plan(49152, 1, 2048, 256, flags=3 << 12) == auto                            # 3 lanes: not a width, ignored
    assert sk.plan_flags(sk.SK_PLAN_LDG, 8) == (1 << 8) | (8 << 12) and sk.plan_flags(sk.SK_PLAN_NO_TMAP) == 1 << 9
    sk.plan_override(sk.SK_PLAN_LDG, 4)                      # the Python-side default for calls made through the binding
    try:
        assert sk.sk_frame_plan(49152, 1, 2048, 256)[0] == 4
    finally:
        sk.plan_override(0, 0)
    assert sk.sk_frame_plan(49152, 1, 2048, 256) == auto


def test_version_and_strerror(sk):
    assert sk.sk_version() >= 100
    assert sk.sk_strerror(0) == "ok"
    for code in (-1, -2, -3, -4, -5, -6):
        assert sk.sk_strerror(code) not in ("ok", "unknown error")
    assert sk.sk_strerror(-99) == "unknown error"


def test_argument_errors_need_no_device(sk):
    L = sk.lib()
    one = C.c_void_p(16)               # never dereferenced: every call below fails validation first
    assert L.sk_power_sums(None, 8, 1, 16, 4, one, one, None) == -1
    assert L.sk_power_sums(one, 8, 1, 16, 1, one, one, None) == -3
    assert L.sk_power_sums(one, 8, 1, 16, 70000, one, one, None) == -3
    assert L.sk_power_sums(one, 9, 1, 16, 4, one, one, None) == -2
    assert L.sk_power_sums(one, 0, 1, 16, 4, one, one, None) == -2
    assert L.sk_combine(one, one, 2, 1, 16, 4, None, 17, one, None) == -4
    assert L.sk_combine(one, one, 2, 1, 16, 4, None, 0, one, None) == -4
    assert L.sk_flag(one, 2, 1, 4, 0, 3.0, 1.0, one, None) == -4
    assert L.sk_flag(one, 2, 1, 4, 16, float("inf"), 1.0, one, None) == -5
    assert L.sk_frame(one, 8, 1, 16, 4, None, 16, 3.0, 1.0, 0, one, one, None, None, None, 0, None) == -6
    assert L.sk_frame(one, 8, 1, 16, 4, None, 16, 3.0, 1.0, 0, one, None, None, None, one, 1 << 20, None) == -1
    assert L.sk_frame(one, 8, 1, 16, 4, None, 16, 3.0, 1.0, 0, one, one, one, None, one, 1 << 20, None) == -1


def test_workspace_bytes(sk):
    # cells * ceil(E/16) doubles (room for the narrowest slabs any plan uses) + cells counters:
    # a function of the shape only, never of the device
    assert sk.sk_frame_workspace_bytes(49152, 1, 2048, 256) == 192 * 128 * 8 + 192 * 4
    assert sk.sk_frame_workspace_bytes(4096, 1, 256, 256) == 16 * 16 * 8 + 16 * 4
    assert sk.sk_frame_workspace_bytes(64, 2, 48, 32) == 4 * 3 * 8 + 4 * 4
    assert sk.sk_frame_workspace_bytes(10, 1, 16, 4) == 0                        # T % M != 0


def test_no_cpu_fallback(sk):
    import torch
    with pytest.raises(sk.SKError):
        sk.sk_frame(torch.zeros(8, 1, 16, dtype=torch.uint8), 4)
    with pytest.raises(sk.SKError):
        sk.sk_power_sums(torch.zeros(8, 1, 16, dtype=torch.uint8), 4)


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle, nor the oracle through the product."""
    bad = re.compile(r"(import\s+oracle|from\s+oracle|from\s+\.+oracle|sk_oracle|libsk_oracle|#include\s*[\"<][^\n]*oracle)")
    pkg = os.path.join(ROOT, "paper_1808_10365_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                assert not bad.search(open(os.path.join(dirpath, fn)).read()), fn
    assert not bad.search(open(os.path.join(ROOT, "include", "sk_b200.h")).read())
    bad2 = re.compile(r"(import\s+paper_1808_10365_b200|from\s+paper_1808_10365_b200|sk_b200\.h|sk_device|sk_kernels|libsk_b200)")
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp", ".c", ".h")):
            assert not bad2.search(open(os.path.join(ROOT, "oracle", fn)).read()), fn
