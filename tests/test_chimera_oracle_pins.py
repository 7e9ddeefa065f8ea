"""Pins of the chimera oracle (the CUDA path is tested in test_gpu_parity.py).

oracle/chimera_oracle.py holds two independent computations: the definition (enumeration) and the
paper's group tensor network.  Here the second is pinned to the first on every
shape enumeration reaches, and to what the mathematics fixes beyond that.
"""
import numpy as np
import pytest

from oracle import chimera_oracle as co
from ttn_inputs import make_chimera_instance


def _rand(M, N, T, rng, lo=-2, hi=3):
    K = rng.integers(lo, hi, size=(M, N, T, T)).astype(np.float64)
    Jv = rng.integers(lo, hi, size=(max(M - 1, 0), N, T)).astype(np.float64)
    Jh = rng.integers(lo, hi, size=(M, max(N - 1, 0), T)).astype(np.float64)
    return K, Jv, Jh


# shapes with <= 20 spins: one K_{4,4} cell, two cells either way, 2 x 2 cells of K_{2,2},
# asymmetric strips of small cells (a transposed index or a swapped Jv / Jh fails one of them)
SHAPES = [(1, 1, 4), (1, 2, 4), (2, 1, 4), (2, 2, 2), (3, 1, 2), (1, 3, 2), (3, 2, 1), (2, 3, 1), (2, 2, 1)]


@pytest.mark.parametrize("M,N,T", SHAPES)
def test_dp_equals_enumeration_integer_couplings(M, N, T):
    rng = np.random.default_rng(100 * M + 10 * N + T)
    for trial in range(3):
        K, Jv, Jh = _rand(M, N, T, rng)
        assert co.dp_chimera(M, N, T, K, Jv, Jh) == co.brute_chimera(M, N, T, K, Jv, Jh)


@pytest.mark.parametrize("M,N,T", [(1, 2, 4), (2, 1, 4), (2, 2, 2), (2, 3, 1)])
def test_dp_equals_enumeration_with_fields(M, N, T):
    rng = np.random.default_rng(7 + M + 3 * N + T)
    K, Jv, Jh = _rand(M, N, T, rng)
    hv = rng.integers(-1, 2, size=(M, N, T)).astype(np.float64)
    hu = rng.integers(-1, 2, size=(M, N, T)).astype(np.float64)
    assert co.dp_chimera(M, N, T, K, Jv, Jh, hv, hu) == co.brute_chimera(M, N, T, K, Jv, Jh, hv, hu)


@pytest.mark.parametrize("M,N,T", [(2, 2, 2), (1, 2, 4)])
def test_dp_equals_enumeration_seeded_pmj(M, N, T):
    for seed in (6000, 6001, 6002):
        I = make_chimera_instance(M, N, seed, T)
        E, g = co.dp_chimera(M, N, T, I.K, I.Jv, I.Jh)
        assert (E, g) == co.brute_chimera(M, N, T, I.K, I.Jv, I.Jh)
        assert g % 2 == 0                                       # global flip, h = 0


@pytest.mark.parametrize("M,N", [(2, 2), (3, 3), (4, 3), (3, 4)])
def test_ferromagnet_and_antiferromagnet_closed_form(M, N):
    """All J = +1: E0 = -#edges, g = 2; the chimera graph is bipartite, so all J = -1 gives the same."""
    T = 4
    ne = co.n_edges(M, N, T)
    assert ne == 16 * M * N + 4 * (M - 1) * N + 4 * M * (N - 1)
    for sgn in (1.0, -1.0):
        K = sgn * np.ones((M, N, T, T)); Jv = sgn * np.ones((M - 1, N, T)); Jh = sgn * np.ones((M, N - 1, T))
        assert co.dp_chimera(M, N, T, K, Jv, Jh) == (-float(ne), 2)


def test_free_and_decoupled_closed_forms():
    M, N, T = 2, 3, 4
    z = lambda *s: np.zeros(s)
    # no couplings at all: every configuration is a ground state
    assert co.dp_chimera(M, N, T, z(M, N, T, T), z(M - 1, N, T), z(M, N - 1, T)) == (0.0, 2 ** (2 * T * M * N))
    # only inter-cell couplings: N T vertical + M T horizontal independent open chains, each with
    # E = -sum|J| and g = 2
    rng = np.random.default_rng(5)
    Jv = rng.choice([-1.0, 1.0], size=(M - 1, N, T)); Jh = rng.choice([-1.0, 1.0], size=(M, N - 1, T))
    E, g = co.dp_chimera(M, N, T, z(M, N, T, T), Jv, Jh)
    assert E == -(np.abs(Jv).sum() + np.abs(Jh).sum())
    assert g == 2 ** (N * T + M * T)
    # fields only: E0 = -sum|h|, g = 2^(#zero fields)
    hv = rng.integers(-1, 2, size=(M, N, T)).astype(np.float64); hu = rng.integers(-1, 2, size=(M, N, T)).astype(np.float64)
    E, g = co.dp_chimera(M, N, T, z(M, N, T, T), z(M - 1, N, T), z(M, N - 1, T), hv, hu)
    assert E == -(np.abs(hv).sum() + np.abs(hu).sum())
    assert g == 2 ** int((hv == 0).sum() + (hu == 0).sum())
    # counts that do not fit int64 are refused, not wrapped (3 x 3 free cells: 2^72 states)
    with pytest.raises(OverflowError):
        co.dp_chimera(3, 3, T, z(3, 3, T, T), z(2, 3, T), z(3, 2, T))


def test_gauge_and_scaling_invariance_beyond_enumeration():
    """3 x 3 cells of K_{4,4} (72 spins): J'_ij = J_ij eps_i eps_j leaves (E0, g) unchanged; a planted
    instance (gauge-transformed ferromagnet) has E0 = -#edges, g = 2; doubling J doubles E0."""
    M, N, T = 3, 3, 4
    I = make_chimera_instance(M, N, 6100, T)
    rng = np.random.default_rng(11)
    ev = rng.choice([-1.0, 1.0], size=(M, N, T)); eu = rng.choice([-1.0, 1.0], size=(M, N, T))
    E, g = co.dp_chimera(M, N, T, I.K, I.Jv, I.Jh)
    assert g % 2 == 0 and E == int(E) and -co.n_edges(M, N, T) <= E < 0
    K2, Jv2, Jh2 = co.gauge(M, N, T, I.K, I.Jv, I.Jh, ev, eu)
    assert co.dp_chimera(M, N, T, K2, Jv2, Jh2) == (E, g)
    assert co.dp_chimera(M, N, T, 2 * I.K, 2 * I.Jv, 2 * I.Jh) == (2 * E, g)
    one = lambda *s: np.ones(s)
    Kp, Jvp, Jhp = co.gauge(M, N, T, one(M, N, T, T), one(M - 1, N, T), one(M, N - 1, T), ev, eu)
    assert co.dp_chimera(M, N, T, Kp, Jvp, Jhp) == (-float(co.n_edges(M, N, T)), 2)


def test_transpose_symmetry():
    """Swapping the roles of rows and columns (and of the two groups of every cell) is a graph
    isomorphism: (M, N, K, Jv, Jh) -> (N, M, K^T per cell and transposed grid, Jh^T, Jv^T)."""
    M, N, T = 2, 3, 4
    I = make_chimera_instance(M, N, 6200, T)
    Kt = np.transpose(I.K, (1, 0, 3, 2)).copy()
    Jvt = np.transpose(I.Jh, (1, 0, 2)).copy()          # [N-1, M, T]
    Jht = np.transpose(I.Jv, (1, 0, 2)).copy()          # [N, M-1, T]
    assert co.dp_chimera(M, N, T, I.K, I.Jv, I.Jh) == co.dp_chimera(N, M, T, Kt, Jvt, Jht)
