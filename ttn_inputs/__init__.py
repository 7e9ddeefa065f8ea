"""Seeded synthetic spin-glass instances (SURVEY.md 8d "Instance generator").

This module holds NONE of the method's arithmetic: it only draws couplings.  It is the one
piece shared, as *data*, by the CUDA path's callers (tests, bench.py) and the CPU oracle.

Generator: SplitMix64 used as a counter-based generator, ``u_i = mix(seed + (i+1)*GAMMA)``.
Draw order: Jh row-major, then Jv row-major, then h row-major.
  * +-J (p = 0.5): +1 if the top bit of the draw is 1, else -1            ("+-J")
  * Gaussian: Box-Muller in float64 from two 53-bit uniforms, scaled, ROUNDED TO float32
    ("Gaussian random couplings and fields"; J ~ N(0,1),
    h ~ N(0, sigma=0.1)).  The oracle receives those float32 values widened to float64.

The paper measures on no public data set: all its instances are random draws
(PAPER.md:124, 282, 302), so these seeded draws are the workload itself.

Layouts: Jh[b][L][L-1], Jv[b][L-1][L], h[b][L][L], float32, C order.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, n: int) -> np.ndarray:
    """First n outputs of SplitMix64 started at `seed` (uint64 array)."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + _GAMMA * np.arange(1, n + 1, dtype=np.uint64)
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def _pm_one(u: np.ndarray) -> np.ndarray:
    return np.where((u >> np.uint64(63)) == 1, 1.0, -1.0).astype(np.float32)


def _gauss(u: np.ndarray, sigma: float) -> np.ndarray:
    """Box-Muller: consumes two draws per value."""
    a = ((u[0::2] >> np.uint64(11)).astype(np.float64) + 1.0) / 9007199254740992.0  # (0,1]
    b = (u[1::2] >> np.uint64(11)).astype(np.float64) / 9007199254740992.0          # [0,1)
    z = np.sqrt(-2.0 * np.log(a)) * np.cos(2.0 * np.pi * b)
    return (sigma * z).astype(np.float32)


@dataclass
class Instance:
    q: int                      # 2 = Ising, 3 = Potts
    L: int
    Jh: np.ndarray              # float32 [L, L-1]
    Jv: np.ndarray              # float32 [L-1, L]
    h: Optional[np.ndarray]     # float32 [L, L] or None
    seed: int
    kind: str


def make_instance(L: int, seed: int, kind: str = "pmj", fields: bool = False, q: int = 2,
                  sigma_j: float = 1.0, sigma_h: float = 0.1) -> Instance:
    """kind: 'pmj' (+-1, p=0.5) or 'gauss' (N(0,sigma_j); fields N(0,sigma_h))."""
    nh, nv, nf = L * (L - 1), (L - 1) * L, (L * L if fields else 0)
    if kind == "pmj":
        u = splitmix64(seed, nh + nv + nf)
        vals = _pm_one(u)
    elif kind == "gauss":
        u = splitmix64(seed, 2 * (nh + nv + nf))
        vals = np.concatenate([_gauss(u[: 2 * (nh + nv)], sigma_j),
                               _gauss(u[2 * (nh + nv):], sigma_h)])
    else:
        raise ValueError(kind)
    Jh = vals[:nh].reshape(L, L - 1).copy()
    Jv = vals[nh:nh + nv].reshape(L - 1, L).copy()
    h = vals[nh + nv:].reshape(L, L).copy() if fields else None
    return Instance(q=q, L=L, Jh=Jh, Jv=Jv, h=h, seed=seed, kind=kind)


def make_batch(L: int, seeds, kind: str = "pmj", fields: bool = False, q: int = 2):
    """Batch-major stacked arrays (Jh[b,L,L-1], Jv[b,L-1,L], h[b,L,L] or None)."""
    inst = [make_instance(L, s, kind, fields, q) for s in seeds]
    Jh = np.stack([i.Jh for i in inst]).astype(np.float32)
    Jv = np.stack([i.Jv for i in inst]).astype(np.float32)
    h = np.stack([i.h for i in inst]).astype(np.float32) if fields else None
    return Jh, Jv, h


# The five BASELINE.json configs.  seed = 1000*cfg + instance.
CONFIGS = {
    1: dict(q=2, L=4, kind="pmj", fields=False, seeds=range(1000, 1032), call="count"),
    2: dict(q=2, L=16, kind="gauss", fields=True, seeds=range(2000, 2256), call="config"),
    3: dict(q=2, L=24, kind="pmj", fields=False, seeds=range(3000, 3016), call="count"),
    4: dict(q=2, L=32, kind="pmj", fields=False, seeds=range(4000, 4001), call="energy"),
    5: dict(q=3, L=18, kind="pmj", fields=False, seeds=range(5000, 5004), call="count"),
}


def config_batch(cfg: int, L: Optional[int] = None, n: Optional[int] = None):
    """Arrays for config `cfg`, optionally at another L (same distribution) / first n seeds."""
    c = CONFIGS[cfg]
    seeds = list(c["seeds"])
    if n is not None:
        seeds = seeds[:n]
    return make_batch(L or c["L"], seeds, c["kind"], c["fields"], c["q"])


@dataclass
class ChimeraInstance:
    M: int                      # rows of unit cells
    N: int                      # columns of unit cells
    T: int                      # spins per group (4 = the D-Wave chimera cell K_{4,4})
    K: np.ndarray               # float32 [M, N, T, T]   vertical-group spin k x horizontal-group spin l
    Jv: np.ndarray              # float32 [M-1, N, T]    vertical group of (r, c) - vertical group of (r+1, c)
    Jh: np.ndarray              # float32 [M, N-1, T]    horizontal group of (r, c) - horizontal group of (r, c+1)
    seed: int


def make_chimera_instance(M: int, N: int, seed: int, T: int = 4) -> ChimeraInstance:
    """+-J (p = 0.5), no field, on the chimera graph of M x N unit cells (SURVEY.md
    8f NEXT-3).  Draw order: K row-major, then Jv, then Jh."""
    nk, nv, nh = M * N * T * T, (M - 1) * N * T, M * (N - 1) * T
    vals = _pm_one(splitmix64(seed, nk + nv + nh))
    return ChimeraInstance(M=M, N=N, T=T, K=vals[:nk].reshape(M, N, T, T).copy(),
                           Jv=vals[nk:nk + nv].reshape(M - 1, N, T).copy(),
                           Jh=vals[nk + nv:].reshape(M, N - 1, T).copy(), seed=seed)
