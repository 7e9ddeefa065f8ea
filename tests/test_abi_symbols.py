"""The C-ABI library builds, loads without a GPU and exports every symbol include/ttn.h declares."""
import ctypes
import os
import re

import pytest

import paper_2008_06888_b200 as ttn

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "ttn.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ttn_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    lib = ttn.lib()
    names = declared_symbols()
    assert set(names) == set(ttn.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n


def test_workspace_bytes_and_argument_errors_without_gpu():
    # 2^32 f32 state = 16 GiB + tables
    n = ttn.workspace_bytes(2, 32, ttn.TROPICAL_F32, 1)
    assert 16 * 2**30 <= n < 16 * 2**30 + 2**26
    n = ttn.workspace_bytes(2, 24, ttn.COUNTING_F32_F64, 16)
    assert n >= 16 * 2**24 * 12
    n = ttn.workspace_bytes(2, 16, ttn.TROPICAL_F32, 256, True)
    assert n >= 256 * 17 * 2**16 * 4
    n = ttn.workspace_bytes(3, 18, ttn.COUNTING_F32_F64, 1)
    assert 3**17 * 12 <= n < 3**17 * 12 + 2**26          # Potts runs on the colour-rotation-reduced third (3^17 elements)
    # h = 0: the flip-reduced half-state suffices (ttn_workspace_bytes_h0)
    n = ttn.workspace_bytes(2, 32, ttn.TROPICAL_F32, 1, h_zero=True)
    assert 8 * 2**30 <= n < 8 * 2**30 + 2**26
    lib = ttn.lib()
    assert lib.ttn_workspace_bytes(5, 8, 0, 1, 0) == 0
    assert lib.ttn_workspace_bytes(2, 0, 0, 1, 0) == 0
    assert lib.ttn_workspace_bytes(2, 40, 0, 1, 0) == 0
    assert lib.ttn_workspace_bytes(3, 21, 0, 1, 0) == 0
    assert lib.ttn_workspace_bytes(2, 8, 0, 0, 0) == 0
    # NULL arguments are rejected before any CUDA call
    e0 = (ctypes.c_double * 1)()
    st = lib.ttn_sweep_energy(4, None, None, None, 1, None, 0, None, e0)
    assert st == 1 and b"NULL" in lib.ttn_last_error()
    assert lib.ttn_version() >= 100


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np
    with pytest.raises(ttn.TTNError):
        ttn.sweep_energy(np.ones((3, 2)), np.ones((2, 3)))


def test_plan_describe_limits_follow_the_call_kind():
    """ttn_plan_describe applies the limits ttn_plan_create applies: counting and config stop at L = 32 for the
    plain and the *_Z2 kinds alike, and the flip-reduced kinds are Ising calls."""
    lib = ttn.lib()
    buf = ctypes.create_string_buffer(16)
    assert lib.ttn_plan_describe(2, 33, ttn.CALL_ENERGY_Z2, buf, 16) > 0          # energy: L <= 34
    for call in (ttn.CALL_COUNT, ttn.CALL_COUNT_Z2, ttn.CALL_CONFIG, ttn.CALL_CONFIG_Z2):
        assert lib.ttn_plan_describe(2, 33, call, buf, 16) == -1, call
        assert lib.ttn_plan_describe(2, 20, call, buf, 16) > 0, call
    for call in (ttn.CALL_ENERGY_Z2, ttn.CALL_COUNT_Z2, ttn.CALL_ENERGY_I16_Z2, ttn.CALL_CONFIG_Z2, ttn.CALL_ENERGY_I16, ttn.CALL_CONFIG):
        assert lib.ttn_plan_describe(3, 8, call, buf, 16) == -1, call
    assert lib.ttn_plan_describe(3, 8, ttn.CALL_COUNT, buf, 16) > 0
    assert lib.ttn_plan_describe(2, 8, 99, buf, 16) == -1


def test_debug_switches_need_the_opt_in(monkeypatch):
    """A stray TTN_DEBUG_* variable changes nothing unless TTN_ENABLE_DEBUG=1 is set too (conftest.py sets it)."""
    half = ttn.workspace_bytes(2, 20, ttn.TROPICAL_F32, 1, h_zero=True)
    full = ttn.workspace_bytes(2, 20, ttn.TROPICAL_F32, 1)
    assert half < full
    monkeypatch.setenv("TTN_DEBUG_Z2", "0")
    assert ttn.workspace_bytes(2, 20, ttn.TROPICAL_F32, 1, h_zero=True) == full     # opted in: the switch acts
    monkeypatch.delenv("TTN_ENABLE_DEBUG")
    assert ttn.workspace_bytes(2, 20, ttn.TROPICAL_F32, 1, h_zero=True) == half     # not opted in: ignored
    monkeypatch.setenv("TTN_DEBUG_FUSED", "0")
    assert ttn.workspace_bytes(2, 20, ttn.TROPICAL_F32, 1) == full
    # the chimera layouts do not depend on TTN_DEBUG_FUSED even when opted in (their gate rows always run fused)
    monkeypatch.setenv("TTN_ENABLE_DEBUG", "1")
    a = ttn.chimera_workspace_bytes(4, 3), ttn.chimera_count_workspace_bytes(3, 3)
    monkeypatch.delenv("TTN_DEBUG_FUSED")
    monkeypatch.delenv("TTN_DEBUG_Z2")
    assert a == (ttn.chimera_workspace_bytes(4, 3), ttn.chimera_count_workspace_bytes(3, 3))
