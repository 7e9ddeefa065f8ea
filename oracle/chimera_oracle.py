"""CPU oracle for the chimera-graph spin glass -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module.
It shares no code with the CUDA path (csrc/ttn_chimera.cuh works on single spins with an ancilla;
this file contracts the paper's group tensors) and was committed, pinned
(tests/test_chimera_oracle_pins.py), before that kernel.

The model ("+-J coupling and no external field on the chimera graph ... unit cells
arranged in a square grid ... Each unit cell contains 8 spins forming a complete bipartite graph.
Each group of four spins within the unit cell connects horizontally or vertically to the spins in
the neighboring unit cells"), energy as Eq. (1):  E = - sum_<ij> J_ij s_i s_j - sum h_i s_i.

    M x N cells, T spins per group (T = 4 on the device; smaller T only so that brute force reaches
    2 x 2 cells).  Cell (r, c) holds a VERTICAL group v[0..T) and a HORIZONTAL group u[0..T).
      K [M][N][T][T]   K[r][c][k][l] couples v_k and u_l of the same cell     (the black tensor)
      Jv[M-1][N][T]    couples v_k of (r, c) with v_k of (r+1, c)             (red squares)
      Jh[M][N-1][T]    couples u_l of (r, c) with u_l of (r, c+1)             (blue squares)
      hv, hu [M][N][T] optional fields on the two groups
    A group value g in [0, 2^T) encodes spins s_k = +1 if bit k of g is 0 else -1.

Two independent computations:
  * brute_chimera: the definition, all 2^(2 T M N) configurations (<= 24 spins).
  * dp_chimera: the paper's tensor network (Fig. 2b): every group is one index of
    dimension 2^T, "these tensors are all 16 x 16 tropical matrices", contracted as the evolution
    of a state of dimension (2^T)^M column by column -- for every column: the horizontal matrices
    H_r[u, u'] act on the M indices, then the column's vertical chain (black tensors K_r[u', v]
    and red matrices V_r[v, v']) is contracted for every boundary value.  CountingTropical
    arithmetic (Eq. (4)): (x, n) (+) = max with counts added on ties, (x) = (x1+x2, n1*n2).
    Values in float64 (exact for integer couplings), counts in int64; OverflowError instead of a
    wrapped count (a later 16-term sum of counts below 2^57 stays below 2^62).
"""
from __future__ import annotations

from typing import Tuple

import numpy as np


def _spins(T: int) -> np.ndarray:
    """spins[g, k] = +1 if bit k of g is 0 else -1."""
    g = np.arange(1 << T)
    return 1.0 - 2.0 * ((g[:, None] >> np.arange(T)[None, :]) & 1)


def n_edges(M: int, N: int, T: int) -> int:
    return M * N * T * T + (M - 1) * N * T + M * (N - 1) * T


def brute_chimera(M, N, T, K, Jv, Jh, hv=None, hu=None) -> Tuple[float, int]:
    """(E0, degeneracy) by enumeration.  Spin id = ((r N + c) 2 + grp) T + k, grp 0 = v, 1 = u."""
    ns = 2 * T * M * N
    assert ns <= 24, "brute force is for tiny instances"
    sid = lambda r, c, grp, k: ((r * N + c) * 2 + grp) * T + k
    edges, fields = [], []
    for r in range(M):
        for c in range(N):
            for k in range(T):
                for l in range(T):
                    edges.append((sid(r, c, 0, k), sid(r, c, 1, l), float(K[r][c][k][l])))
                if r + 1 < M:
                    edges.append((sid(r, c, 0, k), sid(r + 1, c, 0, k), float(Jv[r][c][k])))
                if c + 1 < N:
                    edges.append((sid(r, c, 1, k), sid(r, c + 1, 1, k), float(Jh[r][c][k])))
                if hv is not None:
                    fields.append((sid(r, c, 0, k), float(hv[r][c][k])))
                if hu is not None:
                    fields.append((sid(r, c, 1, k), float(hu[r][c][k])))
    assert len(edges) == n_edges(M, N, T)
    best, cnt = None, 0
    chunk = 1 << min(ns, 16)
    for base in range(0, 1 << ns, chunk):
        conf = np.arange(base, base + chunk, dtype=np.int64)
        s = 1.0 - 2.0 * ((conf[:, None] >> np.arange(ns)[None, :]) & 1)
        e = np.zeros(chunk)
        for i, j, J in edges:
            e -= J * s[:, i] * s[:, j]
        for i, h in fields:
            e -= h * s[:, i]
        m = e.min()
        if best is None or m < best:
            best, cnt = m, int((e == m).sum())
        elif m == best:
            cnt += int((e == m).sum())
    return float(best), cnt


def _matvec(x, n, axis, W):
    """Counting-tropical product of the state (x, n) with the matrix W[old, new] on `axis`."""
    x = np.moveaxis(x, axis, -1)
    n = np.moveaxis(n, axis, -1)
    cand = x[..., :, None] + W                    # [..., old, new]
    m = cand.max(axis=-2)
    nn = (n[..., :, None] * (cand == m[..., None, :])).sum(axis=-2)
    return np.moveaxis(m, -1, axis), np.moveaxis(nn, -1, axis)


def dp_chimera(M, N, T, K, Jv, Jh, hv=None, hu=None) -> Tuple[float, int]:
    """(E0, degeneracy) by the column-by-column contraction of the group tensor network."""
    D = 1 << T
    assert D ** (M + 1) <= 1 << 28, "oracle sizes only"             # 6 x N cells of K_{4,4}: a few GB and minutes
    S = _spins(T)                                                   # [D, T]
    K = np.asarray(K, dtype=np.float64).reshape(M, N, T, T)
    Jv = np.asarray(Jv, dtype=np.float64).reshape(max(M - 1, 0), N, T)
    Jh = np.asarray(Jh, dtype=np.float64).reshape(M, max(N - 1, 0), T)
    zero = np.zeros((M, N, T))
    hv = zero if hv is None else np.asarray(hv, dtype=np.float64).reshape(M, N, T)
    hu = zero if hu is None else np.asarray(hu, dtype=np.float64).reshape(M, N, T)
    # state over the horizontal groups of the current column: F[u^0, ..., u^{M-1}]
    Fx = np.zeros((D,) * M)                                          # tropical one
    Fn = np.ones((D,) * M, dtype=np.int64)
    for c in range(N):
        if c > 0:                                                    # blue squares: H_r[u, u']
            for r in range(M):
                H = (S * Jh[r, c - 1][None, :]) @ S.T                # sum_l J_l s_l(u) s_l(u')
                Fx, Fn = _matvec(Fx, Fn, r, H)
        # the column's vertical chain for every boundary value: G[u^0..u^{M-1}]
        Gx = Gn = None
        for r in range(M):
            # black tensor with the fields of the cell: B[u, v]
            B = (S @ K[r, c].T) @ S.T                                # B[u, v] = sum_kl K[k][l] s_k(v) s_l(u)
            B = B + (S @ hu[r, c])[:, None] + (S @ hv[r, c])[None, :]
            if r == 0:
                Gx, Gn = B.copy(), np.ones_like(B, dtype=np.int64)   # [u^0, v^0]
            else:
                V = (S * Jv[r - 1, c][None, :]) @ S.T                # red matrix V[v, v']
                Gx, Gn = _matvec(Gx, Gn, Gx.ndim - 1, V)             # v^{r-1} -> v^r
                Gx = Gx[..., None, :] + B                            # new index u^r in front of v^r
                Gn = np.broadcast_to(Gn[..., None, :], Gx.shape).copy()
        m = Gx.max(axis=-1)                                          # close the chain: (+) over v^{M-1}
        Gn = (Gn * (Gx == m[..., None])).sum(axis=-1)
        # int64 counts: refuse instead of wrapping (the float64 product sees the magnitude)
        if (Fn.astype(np.float64) * Gn.astype(np.float64)).max() >= 2.0 ** 57:
            raise OverflowError("degeneracy beyond the oracle's int64 range")
        Fx, Fn = Fx + m, Fn * Gn                                     # (x) with the boundary state
    best = Fx.max()
    top = Fn[Fx == best]
    if top.astype(np.float64).sum() >= 2.0 ** 62:
        raise OverflowError("degeneracy beyond the oracle's int64 range")
    return float(-best), int(top.sum())


def gauge(M, N, T, K, Jv, Jh, eps_v, eps_u):
    """J'_ij = J_ij eps_i eps_j for eps in {+-1}: E0 and g are invariant."""
    K2 = np.asarray(K, dtype=np.float64) * eps_v[:, :, :, None] * eps_u[:, :, None, :]
    Jv2 = np.asarray(Jv, dtype=np.float64) * eps_v[:-1] * eps_v[1:]
    Jh2 = np.asarray(Jh, dtype=np.float64) * eps_u[:, :-1] * eps_u[:, 1:]
    return K2, Jv2, Jh2
