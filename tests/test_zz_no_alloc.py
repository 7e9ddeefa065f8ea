"""ttn_sweep_energy_noalloc: the energy sweep for callers that cannot allocate device memory.

Who that is: code that runs inside somebody else's process on somebody else's terms -- a plug-in or
callback in an application whose memory pool has already taken the whole GPU (a raw cudaMalloc fails
there, and the plug-in cannot reach the pool), or a loop that must never meet the device-wide
synchronisation cudaMalloc / cudaFree bring.  For them the library carries a fixed 4.5 MiB scratch
array of its own (include/ttn.h, TTN_NOALLOC_SCRATCH_BYTES) and this one call sweeps inside it.

What is checked here: the call returns what the ordinary workspace call (ttn_sweep_energy, parity-tested
against the oracle in test_gpu_parity.py) returns, on calls made back to back on the shared array --
a large lattice first, so that the smaller sweeps after it run over its left-overs -- and sizes beyond
the array are refused with a message instead of overrunning it.

This file sorts last on purpose: pytest -x stops at the first failure, so a problem here cannot hide a
result of the parity suite.  It passes alone in a fresh process (its first call does the per-device
address look-up) and after the other tests.
"""
import numpy as np
import pytest

import paper_2008_06888_b200 as ttn
from ttn_inputs import make_batch


@pytest.mark.gpu
def test_noalloc_equals_workspace_path_on_consecutive_calls():
    # call 1: one 20x20 lattice, Gaussian couplings and fields -- the full 2^20 state, 4.07 of the 4.5 MiB
    L = 20
    Jh, Jv, h = make_batch(L, [7100], "gauss", fields=True)
    E_ws = ttn.sweep_energy(Jh, Jv, h)
    E_na = ttn.sweep_energy_noalloc(Jh, Jv, h)
    assert abs(E_na[0] - E_ws[0]) <= 1e-5 * abs(E_ws[0]), (E_na, E_ws)     # the f32 tolerance of the parity suite
    first = E_na.copy()

    # call 2, straight after, over what call 1 left in the array: a batch of 16x16 +-J lattices without a
    # field (the flip-reduced half-state plan), integer couplings: bit-exact
    L2 = 16
    Jh2, Jv2, _ = make_batch(L2, [7200 + i for i in range(8)], "pmj")
    E_ws2 = ttn.sweep_energy(Jh2, Jv2)
    E_na2 = ttn.sweep_energy_noalloc(Jh2, Jv2)
    assert np.array_equal(E_na2, E_ws2), (E_na2, E_ws2)

    # call 3: a lattice small enough for the generic tile kernel (L < 12), with integer fields
    L3 = 9
    Jh3, Jv3, h3 = make_batch(L3, [7300, 7301], "pmj", fields=True)
    h3 = np.rint(h3 * 10).astype(np.float32)
    assert np.array_equal(ttn.sweep_energy_noalloc(Jh3, Jv3, h3), ttn.sweep_energy(Jh3, Jv3, h3))

    # call 4: the first instance again -- same bits as the first time, whatever the calls between left behind
    again = ttn.sweep_energy_noalloc(Jh, Jv, h)
    assert np.array_equal(again, first), (again, first)

    # degenerate sizes: a single spin, a 2x2 and a 5x5 lattice (batches of 3, integer couplings and fields)
    rng = np.random.default_rng(7350)
    for Ls in (1, 2, 5):
        Jhs = rng.integers(-3, 4, size=(3, Ls, Ls - 1)).astype(np.float32)
        Jvs = rng.integers(-3, 4, size=(3, Ls - 1, Ls)).astype(np.float32)
        hs = rng.integers(-2, 3, size=(3, Ls, Ls)).astype(np.float32)
        assert np.array_equal(ttn.sweep_energy_noalloc(Jhs, Jvs, hs), ttn.sweep_energy(Jhs, Jvs, hs)), Ls

    # the largest field-free lattice that fits (21x21, half-state of 2^20 elements)
    L4 = 21
    Jh4, Jv4, _ = make_batch(L4, [7400], "pmj")
    assert np.array_equal(ttn.sweep_energy_noalloc(Jh4, Jv4), ttn.sweep_energy(Jh4, Jv4))


def _raw_call(L, Jh, Jv, h):
    """The C entry point itself, default stream (the binding asks torch for the current stream, which needs a GPU)."""
    import ctypes
    fp = ctypes.POINTER(ctypes.c_float)
    E0 = np.zeros(Jh.shape[0], dtype=np.float64)
    st = ttn.lib().ttn_sweep_energy_noalloc(L, Jh.ctypes.data_as(fp), Jv.ctypes.data_as(fp), h.ctypes.data_as(fp),
                                            Jh.shape[0], None, E0.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return st, ttn.lib().ttn_last_error().decode()


def test_noalloc_refuses_sizes_beyond_the_array():
    """Refused on the host, before any CUDA call (so this runs without a GPU): 22x22 needs 16 MiB."""
    L = 22
    Jh, Jv, h = make_batch(L, [7500], "pmj", fields=True)
    assert ttn.workspace_bytes(2, L, ttn.TROPICAL_F32, 1) > ttn.NOALLOC_SCRATCH_BYTES
    st, msg = _raw_call(L, Jh, Jv, h)
    assert st == 2 and str(ttn.NOALLOC_SCRATCH_BYTES) in msg, (st, msg)
    # 21x21 fits only without a field
    Jh, Jv, h = make_batch(21, [7501], "pmj", fields=True)
    st, msg = _raw_call(21, Jh, Jv, h)
    assert st == 2 and str(ttn.NOALLOC_SCRATCH_BYTES) in msg, (st, msg)
    # the limits quoted in ttn.h
    assert ttn.workspace_bytes(2, 20, ttn.TROPICAL_F32, 1) <= ttn.NOALLOC_SCRATCH_BYTES
    assert ttn.workspace_bytes(2, 21, ttn.TROPICAL_F32, 1, h_zero=True) <= ttn.NOALLOC_SCRATCH_BYTES
    assert ttn.workspace_bytes(2, 16, ttn.TROPICAL_F32, 14) <= ttn.NOALLOC_SCRATCH_BYTES
