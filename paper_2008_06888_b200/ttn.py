"""Thin Python binding of libttn.so (include/ttn.h).  Argument marshalling only: every step of
the sweep runs in the library's CUDA kernels.  torch is used for the device workspace buffer and
the current stream, nothing else.  There is no CPU fallback: if the library cannot be built or
loaded, or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Tuple

import numpy as np

from .build import build

TROPICAL_F32 = 0
COUNTING_F32_F64 = 1
TROPICAL_I16 = 2
CALL_ENERGY, CALL_COUNT, CALL_CONFIG, CALL_ENERGY_I16 = 0, 1, 2, 3
CALL_ENERGY_Z2, CALL_COUNT_Z2, CALL_ENERGY_I16_Z2, CALL_CONFIG_Z2 = 4, 5, 6, 7      # CALL_ENERGY / CALL_COUNT / CALL_ENERGY_I16 / CALL_CONFIG with the h = 0 flip-reduced half-state required (ttn.h)

EXPORTS = [
    "ttn_workspace_bytes", "ttn_workspace_bytes_h0", "ttn_sweep_energy", "ttn_sweep_energy_i16", "ttn_sweep_count", "ttn_ground_config",
    "ttn_potts3_sweep_energy", "ttn_potts3_sweep_count", "ttn_plan_create", "ttn_plan_launch",
    "ttn_plan_read", "ttn_plan_destroy", "ttn_plan_num_launches", "ttn_plan_num_passes",
    "ttn_plan_describe", "ttn_plan_state_elements", "ttn_last_error", "ttn_version",
    "ttn_chimera_workspace_bytes", "ttn_chimera_sweep_energy_i16",
    "ttn_chimera_count_workspace_bytes", "ttn_chimera_sweep_count",
    "ttn_sweep_energy_noalloc",
]
NOALLOC_SCRATCH_BYTES = 4718592      # TTN_NOALLOC_SCRATCH_BYTES of include/ttn.h

_STATUS = {1: "TTN_EINVAL", 2: "TTN_EUNSUPPORTED", 3: "TTN_ENOMEM", 4: "TTN_ECUDA"}


class TTNError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """Load (building if stale) the C-ABI library.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        fp = ctypes.POINTER(ctypes.c_float)
        dp = ctypes.POINTER(ctypes.c_double)
        i8 = ctypes.POINTER(ctypes.c_int8)
        vp, sz, ci = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int
        L.ttn_workspace_bytes.argtypes = [ci, ci, ci, ci, ci]
        L.ttn_workspace_bytes.restype = sz
        L.ttn_workspace_bytes_h0.argtypes = [ci, ci, ci, ci, ci]
        L.ttn_workspace_bytes_h0.restype = sz
        L.ttn_sweep_energy.argtypes = [ci, fp, fp, fp, ci, vp, sz, vp, dp]
        L.ttn_sweep_energy_i16.argtypes = [ci, fp, fp, fp, ci, vp, sz, vp, dp]
        L.ttn_sweep_energy_noalloc.argtypes = [ci, fp, fp, fp, ci, vp, dp]
        L.ttn_sweep_count.argtypes = [ci, fp, fp, fp, ci, vp, sz, vp, dp, dp]
        L.ttn_ground_config.argtypes = [ci, fp, fp, fp, ci, vp, sz, vp, dp, i8]
        L.ttn_potts3_sweep_energy.argtypes = [ci, fp, fp, ci, vp, sz, vp, dp]
        L.ttn_potts3_sweep_count.argtypes = [ci, fp, fp, ci, vp, sz, vp, dp, dp]
        L.ttn_plan_create.argtypes = [ci, ci, ci, fp, fp, fp, ci, vp, sz, vp, ctypes.POINTER(vp)]
        L.ttn_plan_launch.argtypes = [vp, vp]
        L.ttn_plan_read.argtypes = [vp, vp, dp, dp, i8]
        L.ttn_plan_destroy.argtypes = [vp]
        L.ttn_plan_destroy.restype = None
        L.ttn_plan_num_launches.argtypes = [vp]
        L.ttn_plan_num_passes.argtypes = [vp]
        L.ttn_plan_state_elements.argtypes = [vp]
        L.ttn_plan_state_elements.restype = ctypes.c_ulonglong
        L.ttn_plan_describe.argtypes = [ci, ci, ci, ctypes.c_char_p, sz]
        L.ttn_plan_describe.restype = ctypes.c_long
        L.ttn_last_error.restype = ctypes.c_char_p
        L.ttn_chimera_workspace_bytes.argtypes = [ci, ci]
        L.ttn_chimera_workspace_bytes.restype = sz
        L.ttn_chimera_sweep_energy_i16.argtypes = [ci, ci, fp, fp, fp, vp, sz, vp, dp]
        L.ttn_chimera_count_workspace_bytes.argtypes = [ci, ci]
        L.ttn_chimera_count_workspace_bytes.restype = sz
        L.ttn_chimera_sweep_count.argtypes = [ci, ci, fp, fp, fp, vp, sz, vp, dp, dp]
        _lib = L
    return _lib


def _check(st: int):
    if st != 0:
        raise TTNError(st, lib().ttn_last_error().decode())


def _f32(a, shape, name):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32))
    if a.shape != shape:
        raise ValueError(f"{name}: expected shape {shape}, got {a.shape}")
    return a


def _fptr(a):
    if a is None or a.size == 0:
        return None
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def _couplings(Jh, Jv, h):
    """Accept [L,L-1]/[L-1,L]/[L,L] or batched [B,...]; returns batched float32 arrays."""
    Jv = np.asarray(Jv, dtype=np.float32)
    Jh = np.asarray(Jh, dtype=np.float32)
    if Jv.ndim == 2:
        Jv, Jh = Jv[None], Jh[None]
        h = None if h is None else np.asarray(h, dtype=np.float32)[None]
    B, L = Jv.shape[0], Jv.shape[2]
    Jh = _f32(Jh, (B, L, L - 1), "Jh")
    Jv = _f32(Jv, (B, L - 1, L), "Jv")
    h = None if h is None else _f32(h, (B, L, L), "h")
    return B, L, Jh, Jv, h


def workspace_bytes(q: int, L: int, mode: int, batch: int, want_config: bool = False, h_zero: bool = False) -> int:
    """ttn_workspace_bytes, or ttn_workspace_bytes_h0 when the caller will pass no (or an all-zero) field."""
    fn = lib().ttn_workspace_bytes_h0 if h_zero else lib().ttn_workspace_bytes
    n = int(fn(q, L, mode, batch, int(want_config)))
    if n == 0:
        raise TTNError(2, f"unsupported q={q} L={L} mode={mode} batch={batch}")
    return n


def alloc_workspace(nbytes: int, device="cuda:0"):
    """A torch uint8 tensor used purely as a device buffer."""
    import torch
    if not torch.cuda.is_available():
        raise TTNError(4, "no CUDA device: the tropical sweep has no CPU path")
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def _stream_ptr(stream=None) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def plan_describe(q: int, L: int, call: int) -> str:
    """Text dump of the pass schedule (host only; no device needed)."""
    n = lib().ttn_plan_describe(q, L, call, ctypes.create_string_buffer(1), 1)
    if n < 0:
        raise TTNError(1, f"cannot plan q={q} L={L} call={call}")
    buf = ctypes.create_string_buffer(n + 1)
    lib().ttn_plan_describe(q, L, call, buf, n + 1)
    return buf.value.decode()


class Plan:
    """ttn_plan_* wrapper: upload once, launch (async) many times, read results."""

    def __init__(self, q: int, call: int, Jh, Jv, h=None, workspace=None, stream=None):
        self.B, self.L, self.Jh, self.Jv, self.h = _couplings(Jh, Jv, h)
        self.q, self.call = q, call
        mode = _mode_of(call)
        need = workspace_bytes(q, self.L, mode, self.B, call in (CALL_CONFIG, CALL_CONFIG_Z2), _h_zero(self.h))
        self.workspace = workspace if workspace is not None else alloc_workspace(need)
        if self.workspace.numel() * self.workspace.element_size() < need:
            raise TTNError(3, "workspace too small")
        self._p = ctypes.c_void_p()
        _check(lib().ttn_plan_create(q, self.L, call, _fptr(self.Jh), _fptr(self.Jv), _fptr(self.h),
                                     self.B, self.workspace.data_ptr(),
                                     self.workspace.numel() * self.workspace.element_size(),
                                     _stream_ptr(stream), ctypes.byref(self._p)))

    @property
    def num_launches(self) -> int:
        return int(lib().ttn_plan_num_launches(self._p))

    @property
    def num_passes(self) -> int:
        return int(lib().ttn_plan_num_passes(self._p))

    @property
    def state_elements(self) -> int:
        """Stored state-vector elements per instance (2^(L-1) under the h = 0 flip reduction)."""
        return int(lib().ttn_plan_state_elements(self._p))

    def launch(self, stream=None):
        _check(lib().ttn_plan_launch(self._p, _stream_ptr(stream)))

    def read(self, stream=None):
        E0 = np.zeros(self.B, dtype=np.float64)
        g = np.zeros(self.B, dtype=np.float64) if self.call in (CALL_COUNT, CALL_COUNT_Z2) else None
        sig = np.zeros((self.B, self.L, self.L), dtype=np.int8) if self.call in (CALL_CONFIG, CALL_CONFIG_Z2) else None
        _check(lib().ttn_plan_read(
            self._p, _stream_ptr(stream), E0.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
            g.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if g is not None else None,
            sig.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)) if sig is not None else None))
        return E0, g, sig

    def close(self):
        if self._p:
            lib().ttn_plan_destroy(self._p)
            self._p = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _h_zero(h) -> bool:
    return h is None or not np.any(h)


def _mode_of(call: int) -> int:
    return {CALL_COUNT: COUNTING_F32_F64, CALL_COUNT_Z2: COUNTING_F32_F64, CALL_ENERGY_I16: TROPICAL_I16, CALL_ENERGY_I16_Z2: TROPICAL_I16}.get(call, TROPICAL_F32)


def _one_call(fn_name, q, call, Jh, Jv, h, workspace, stream):
    B, L, Jh, Jv, h = _couplings(Jh, Jv, h)
    mode = _mode_of(call)
    need = workspace_bytes(q, L, mode, B, call == CALL_CONFIG, q == 2 and _h_zero(h))
    ws = workspace if workspace is not None else alloc_workspace(need)
    wsb = ws.numel() * ws.element_size()
    E0 = np.zeros(B, dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    args = [L, _fptr(Jh), _fptr(Jv)]
    if q == 2:
        args.append(_fptr(h))
    args += [B, ws.data_ptr(), wsb, _stream_ptr(stream), E0.ctypes.data_as(dp)]
    extra = None
    if call == CALL_COUNT:
        extra = np.zeros(B, dtype=np.float64)
        args.append(extra.ctypes.data_as(dp))
    elif call == CALL_CONFIG:
        extra = np.zeros((B, L, L), dtype=np.int8)
        args.append(extra.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)))
    _check(getattr(lib(), fn_name)(*args))
    return E0, extra


def sweep_energy(Jh, Jv, h=None, workspace=None, stream=None) -> np.ndarray:
    """ttn_sweep_energy: ground-state energies E0[batch] (Tropical<f32> sweep)."""
    return _one_call("ttn_sweep_energy", 2, CALL_ENERGY, Jh, Jv, h, workspace, stream)[0]


def sweep_energy_noalloc(Jh, Jv, h=None, stream=None) -> np.ndarray:
    """ttn_sweep_energy_noalloc: the E0[batch] of sweep_energy, for callers that cannot allocate device memory
    (a plug-in inside an application whose pool owns the GPU, a loop that must not meet cudaMalloc's
    device-wide synchronisation).  No workspace is passed or allocated: the sweep runs in a
    NOALLOC_SCRATCH_BYTES array built into libttn.so, which bounds the size (one lattice up to L = 20 with a
    field, L = 21 without) and which all calls on a device share -- do not overlap them.  See include/ttn.h."""
    B, L, Jh, Jv, h = _couplings(Jh, Jv, h)
    E0 = np.zeros(B, dtype=np.float64)
    _check(lib().ttn_sweep_energy_noalloc(L, _fptr(Jh), _fptr(Jv), _fptr(h), B, _stream_ptr(stream),
                                          E0.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
    return E0


def sweep_energy_i16(Jh, Jv, h=None, workspace=None, stream=None) -> np.ndarray:
    """ttn_sweep_energy_i16: the same E0[batch] in Tropical<i16> (integer-valued couplings only)."""
    return _one_call("ttn_sweep_energy_i16", 2, CALL_ENERGY_I16, Jh, Jv, h, workspace, stream)[0]


def sweep_count(Jh, Jv, h=None, workspace=None, stream=None) -> Tuple[np.ndarray, np.ndarray]:
    """ttn_sweep_count: (E0[batch], degeneracy[batch]) (CountingTropical sweep)."""
    return _one_call("ttn_sweep_count", 2, CALL_COUNT, Jh, Jv, h, workspace, stream)


def ground_config(Jh, Jv, h=None, workspace=None, stream=None) -> Tuple[np.ndarray, np.ndarray]:
    """ttn_ground_config: (E0[batch], sigma[batch,L,L] of +-1)."""
    return _one_call("ttn_ground_config", 2, CALL_CONFIG, Jh, Jv, h, workspace, stream)


def potts3_sweep_energy(Jh, Jv, workspace=None, stream=None) -> np.ndarray:
    return _one_call("ttn_potts3_sweep_energy", 3, CALL_ENERGY, Jh, Jv, None, workspace, stream)[0]


def potts3_sweep_count(Jh, Jv, workspace=None, stream=None) -> Tuple[np.ndarray, np.ndarray]:
    return _one_call("ttn_potts3_sweep_count", 3, CALL_COUNT, Jh, Jv, None, workspace, stream)


def chimera_workspace_bytes(M: int, N: int) -> int:
    n = lib().ttn_chimera_workspace_bytes(M, N)
    if n == 0:
        raise TTNError(2, f"chimera: unsupported size M={M}, N={N}")
    return n


def chimera_sweep_energy_i16(K, Jv, Jh, workspace=None, stream=None) -> float:
    """ttn_chimera_sweep_energy_i16: ground-state energy of the +-J (integer-coupling) spin glass on
    the chimera graph of M x N unit cells; K[M,N,4,4], Jv[M-1,N,4], Jh[M,N-1,4]."""
    K = np.ascontiguousarray(np.asarray(K, dtype=np.float32))
    if K.ndim != 4 or K.shape[2:] != (4, 4):
        raise ValueError(f"K: expected shape [M, N, 4, 4], got {K.shape}")
    M, N = K.shape[:2]
    Jv = _f32(Jv, (M - 1, N, 4), "Jv")
    Jh = _f32(Jh, (M, N - 1, 4), "Jh")
    need = chimera_workspace_bytes(M, N)
    ws = workspace if workspace is not None else alloc_workspace(need)
    E0 = np.zeros(1, dtype=np.float64)
    _check(lib().ttn_chimera_sweep_energy_i16(M, N, _fptr(K), _fptr(Jv), _fptr(Jh), ws.data_ptr(),
                                              ws.numel() * ws.element_size(), _stream_ptr(stream),
                                              E0.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
    return float(E0[0])


def chimera_count_workspace_bytes(M: int, N: int) -> int:
    n = lib().ttn_chimera_count_workspace_bytes(M, N)
    if n == 0:
        raise TTNError(2, f"chimera: unsupported size M={M}, N={N}")
    return n


def chimera_sweep_count(K, Jv, Jh, workspace=None, stream=None) -> Tuple[float, float]:
    """ttn_chimera_sweep_count: (E0, degeneracy) of the integer-coupling spin glass on the chimera graph."""
    K = np.ascontiguousarray(np.asarray(K, dtype=np.float32))
    if K.ndim != 4 or K.shape[2:] != (4, 4):
        raise ValueError(f"K: expected shape [M, N, 4, 4], got {K.shape}")
    M, N = K.shape[:2]
    Jv = _f32(Jv, (M - 1, N, 4), "Jv")
    Jh = _f32(Jh, (M, N - 1, 4), "Jh")
    need = chimera_count_workspace_bytes(M, N)
    ws = workspace if workspace is not None else alloc_workspace(need)
    E0 = np.zeros(1, dtype=np.float64)
    g = np.zeros(1, dtype=np.float64)
    dp = ctypes.POINTER(ctypes.c_double)
    _check(lib().ttn_chimera_sweep_count(M, N, _fptr(K), _fptr(Jv), _fptr(Jh), ws.data_ptr(),
                                         ws.numel() * ws.element_size(), _stream_ptr(stream),
                                         E0.ctypes.data_as(dp), g.ctypes.data_as(dp)))
    return float(E0[0]), float(g[0])
