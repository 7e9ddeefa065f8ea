"""Pins for the CPU oracle (oracle/ttn_oracle.c) against what the paper and the mathematics fix.

The paper prints no instance-level value, so the pins are: the definition
(Eq. (1)) by enumeration, closed forms, invariants and special cases.  Each is
chosen so a plausible mistake (dropped term, wrong sign/index, transposed operand, wrong tie
rule of Eq. (4)) fails at least one.
"""
import itertools

import numpy as np
import pytest

import oracle
from ttn_inputs import make_instance

RNG = np.random.default_rng(20200806)


def py_brute_ising(L, Jh, Jv, h):
    """Eq. (1) by itertools, pure Python -- independent of the C enumeration."""
    best, cnt = None, 0
    for cfg in itertools.product((1, -1), repeat=L * L):
        s = np.array(cfg).reshape(L, L)
        E = -(Jh * s[:, :-1] * s[:, 1:]).sum() - (Jv * s[:-1, :] * s[1:, :]).sum()
        if h is not None:
            E -= (h * s).sum()
        if best is None or E < best:
            best, cnt = E, 1
        elif E == best:
            cnt += 1
    return float(best), cnt


def rand_int_instance(L, lo=-3, hi=3, fields=True):
    Jh = RNG.integers(lo, hi + 1, size=(L, L - 1)).astype(np.float64)
    Jv = RNG.integers(lo, hi + 1, size=(L - 1, L)).astype(np.float64)
    h = RNG.integers(lo, hi + 1, size=(L, L)).astype(np.float64) if fields else None
    return Jh, Jv, h


# ---------------------------------------------------------------------------- O-brute
@pytest.mark.parametrize("L", [2, 3])
def test_c_brute_equals_python_enumeration(L):
    for fields in (False, True):
        Jh, Jv, h = rand_int_instance(L, fields=fields)
        E_py, g_py = py_brute_ising(L, Jh, Jv, h)
        E_c, g_c, sig = oracle.brute_ising(L, Jh, Jv, h)
        assert E_c == E_py and g_c == g_py
        assert oracle.ising_energy(L, Jh, Jv, h, sig) == E_c


def test_energy_function_hand_example():
    # 2x2, worked by hand from Eq. (1): bonds (00-01)=1, (10-11)=2, (00-10)=3, (01-11)=-1, h=0.5 at (0,0)
    Jh = np.array([[1.0], [2.0]]); Jv = np.array([[3.0, -1.0]])
    h = np.array([[0.5, 0.0], [0.0, 0.0]])
    up = np.ones((2, 2), dtype=np.int8)
    assert oracle.ising_energy(2, Jh, Jv, h, up) == -(1 + 2 + 3 - 1) - 0.5
    s = np.array([[1, -1], [1, 1]], dtype=np.int8)   # flip (0,1): bonds 1 and -1 change sign
    assert oracle.ising_energy(2, Jh, Jv, h, s) == -(-1 + 2 + 3 + 1) - 0.5
    # all bonds satisfied would need s01 = s00 = s10 = s11 = -s01: frustrated.  One of the two
    # weakest bonds (|J| = 1: the +1 or the -1) breaks, s00 aligns with h: E0 = -5.5, g = 2.
    E0, g, _ = oracle.brute_ising(2, Jh, Jv, h)
    assert E0 == -5.5 and g == 2
    assert oracle.dp_ising(2, Jh, Jv, h)[:2] == (-5.5, 2)


# ---------------------------------------------------------------------------- O-dp vs O-brute
@pytest.mark.parametrize("L", [1, 2, 3, 4])
@pytest.mark.parametrize("kind", ["pmj", "int_h", "gauss_h"])
def test_dp_equals_brute_ising(L, kind):
    for rep in range(6 if L < 4 else 3):
        if kind == "pmj":
            inst = make_instance(L, 100 * L + rep, "pmj")
            Jh, Jv, h = inst.Jh, inst.Jv, None
        elif kind == "int_h":
            Jh, Jv, h = rand_int_instance(L)
        else:
            inst = make_instance(L, 777 * L + rep, "gauss", fields=True)
            Jh, Jv, h = inst.Jh, inst.Jv, inst.h
        Eb, gb, sb = oracle.brute_ising(L, Jh, Jv, h)
        Ed, gd, sd = oracle.dp_ising(L, Jh, Jv, h, count=True, config=True)
        if kind == "gauss_h":
            assert abs(Ed - Eb) <= 1e-12 * max(1.0, abs(Eb))
            assert gd == gb == 1
            assert np.array_equal(sd, sb)               # unique ground state
        else:
            assert Ed == Eb and gd == gb                # exact for integers
        assert abs(oracle.ising_energy(L, Jh, Jv, h, sd) - Eb) <= 1e-12 * max(1.0, abs(Eb))
        # energy-only mode agrees
        E2, g2, _ = oracle.dp_ising(L, Jh, Jv, h, count=False)
        assert E2 == Ed and g2 is None


def test_dp_equals_brute_ising_L5():
    inst = make_instance(5, 55, "pmj")
    Eb, gb, _ = oracle.brute_ising(5, inst.Jh, inst.Jv, None)
    Ed, gd, sd = oracle.dp_ising(5, inst.Jh, inst.Jv, None, config=True)
    assert (Ed, gd) == (Eb, gb)
    assert oracle.ising_energy(5, inst.Jh, inst.Jv, None, sd) == Eb


# ---------------------------------------------------------------------------- closed forms
@pytest.mark.parametrize("L", [2, 3, 4, 7, 10, 13])
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_ferromagnet_and_antiferromagnet(L, sign):
    # all J = +1, h = 0: E0 = -#edges = -2L(L-1), g = 2 (north_star); AF is the same by the
    # bipartite gauge.
    Jh = np.full((L, L - 1), sign); Jv = np.full((L - 1, L), sign)
    E0, g, sig = oracle.dp_ising(L, Jh, Jv, None, config=True)
    assert E0 == -2 * L * (L - 1) and g == 2
    if sign > 0:
        assert abs(sig.sum()) == L * L
    else:
        r, c = np.indices((L, L))
        assert abs((sig * (1 - 2 * ((r + c) & 1))).sum()) == L * L


@pytest.mark.parametrize("L", [1, 2, 3, 4, 8, 11])
def test_free_spins_count_is_power_of_two(L):
    Jh = np.zeros((L, max(L - 1, 0))); Jv = np.zeros((max(L - 1, 0), L))
    E0, g, _ = oracle.dp_ising(L, Jh, Jv, None)
    assert E0 == 0.0 and g == 1 << (L * L)         # 2^121 at L = 11: exercises the 128-bit count
    assert np.copysign(1.0, E0) == 1.0             # +0.0, never -0.0


def test_count_overflow_is_trapped():
    L = 12                                          # 2^144 > 2^128
    with pytest.raises(oracle.OracleOverflow):
        oracle.dp_ising(L, np.zeros((L, L - 1)), np.zeros((L - 1, L)), None)


def test_fields_only():
    L = 5
    h = RNG.integers(-2, 3, size=(L, L)).astype(np.float64)
    E0, g, sig = oracle.dp_ising(L, np.zeros((L, L - 1)), np.zeros((L - 1, L)), h, config=True)
    assert E0 == -np.abs(h).sum() and g == 1 << int((h == 0).sum())
    assert np.all(sig[h > 0] == 1) and np.all(sig[h < 0] == -1)   # bit 0 <-> sigma=+1 carries +h (A3)


@pytest.mark.parametrize("L", [3, 6, 9])
def test_decoupled_chains_both_directions(L):
    # Jv = 0: L independent open chains along rows: E0 = -sum|Jh|, g = 2^L.  And the transposed
    # statement with Jh = 0.  Catches a swapped/transposed Jh, Jv operand.
    Jh = RNG.normal(size=(L, L - 1)); Jv = RNG.normal(size=(L - 1, L))
    E0, g, _ = oracle.dp_ising(L, Jh, np.zeros((L - 1, L)), None)
    assert abs(E0 + np.abs(Jh).sum()) < 1e-12 * L * L and g == 1 << L
    E0, g, _ = oracle.dp_ising(L, np.zeros((L, L - 1)), Jv, None)
    assert abs(E0 + np.abs(Jv).sum()) < 1e-12 * L * L and g == 1 << L


def test_single_frustrated_plaquette():
    # 2x2 with three +1 bonds and one -1: one bond must break: E0 = -2, and 4 ways x 2 flips = 8.
    Jh = np.array([[1.0], [1.0]]); Jv = np.array([[1.0, -1.0]])
    E0, g, _ = oracle.dp_ising(2, Jh, Jv, None)
    assert E0 == -2.0 and g == 8


# ---------------------------------------------------------------------------- invariants
@pytest.mark.parametrize("L", [6, 9, 12])
def test_symmetries_pmj(L):
    inst = make_instance(L, 4242 + L, "pmj")
    Jh, Jv = inst.Jh.astype(np.float64), inst.Jv.astype(np.float64)
    E0, g, sig = oracle.dp_ising(L, Jh, Jv, None, config=True)
    assert g % 2 == 0                                   # global flip, h = 0 (north_star)
    assert oracle.ising_energy(L, Jh, Jv, None, sig) == E0
    # transpose: Jh <-> Jv^T   (the algorithm treats the two directions differently, G5)
    assert oracle.dp_ising(L, Jv.T.copy(), Jh.T.copy(), None)[:2] == (E0, g)
    # left-right and up-down reflections
    assert oracle.dp_ising(L, Jh[:, ::-1].copy(), Jv[:, ::-1].copy(), None)[:2] == (E0, g)
    assert oracle.dp_ising(L, Jh[::-1, :].copy(), Jv[::-1, :].copy(), None)[:2] == (E0, g)
    # scaling by 2^k is exact
    assert oracle.dp_ising(L, 8 * Jh, 8 * Jv, None)[:2] == (8 * E0, g)
    # gauge: J'_ij = J_ij e_i e_j leaves E0, g unchanged
    eps = RNG.choice([-1.0, 1.0], size=(L, L))
    Jh2 = Jh * eps[:, :-1] * eps[:, 1:]; Jv2 = Jv * eps[:-1, :] * eps[1:, :]
    E2, g2, sig2 = oracle.dp_ising(L, Jh2, Jv2, None, config=True)
    assert (E2, g2) == (E0, g)
    assert oracle.ising_energy(L, Jh, Jv, None, (sig2 * eps).astype(np.int8)) == E0


def test_gauge_with_fields_maps_configuration():
    L = 7
    inst = make_instance(L, 99, "gauss", fields=True)
    Jh, Jv, h = (a.astype(np.float64) for a in (inst.Jh, inst.Jv, inst.h))
    E0, g, sig = oracle.dp_ising(L, Jh, Jv, h, config=True)
    eps = RNG.choice([-1.0, 1.0], size=(L, L))
    E2, g2, sig2 = oracle.dp_ising(L, Jh * eps[:, :-1] * eps[:, 1:], Jv * eps[:-1, :] * eps[1:, :],
                                   h * eps, config=True)
    assert abs(E2 - E0) < 1e-11 and g == g2 == 1
    assert np.array_equal(sig2 * eps.astype(np.int8), sig)


def test_planted_ground_state():
    # gauge-transformed ferromagnet: looks like +-J disorder, E0 = -2L(L-1), g = 2, sigma* = +-eps
    L = 14
    eps = RNG.choice([-1, 1], size=(L, L))
    Jh = (eps[:, :-1] * eps[:, 1:]).astype(np.float64); Jv = (eps[:-1, :] * eps[1:, :]).astype(np.float64)
    E0, g, sig = oracle.dp_ising(L, Jh, Jv, None, config=True)
    assert E0 == -2 * L * (L - 1) and g == 2
    assert np.array_equal(sig, eps) or np.array_equal(sig, -eps)


@pytest.mark.parametrize("L", [3, 5, 6])
def test_configuration_is_minus_dE0_dh(L):
    # "ground state energy is a piecewise linear function of the fields ... finite-difference of
    # the energy with respect to fields suffices": sigma_i = -dE0/dh_i.
    inst = make_instance(L, 31 + L, "gauss", fields=True)
    Jh, Jv, h = (a.astype(np.float64) for a in (inst.Jh, inst.Jv, inst.h))
    _, _, sig = oracle.dp_ising(L, Jh, Jv, h, config=True)
    d = 1e-6
    for (r, c) in [(0, 0), (L // 2, L // 2), (L - 1, 0), (L - 1, L - 1), (1, L - 2)]:
        hp = h.copy(); hp[r, c] += d
        hm = h.copy(); hm[r, c] -= d
        Ep = oracle.dp_ising(L, Jh, Jv, hp, count=False)[0]
        Em = oracle.dp_ising(L, Jh, Jv, hm, count=False)[0]
        assert abs(-(Ep - Em) / (2 * d) - sig[r, c]) < 1e-4


def test_residual_entropy_sanity():
    # literature value quoted by the paper: s ~ 0.07 for the +-J square lattice;
    # open boundaries and finite L shift it -- wide band, sanity only.
    L = 12
    s = np.mean([np.log(oracle.dp_ising(L, *(lambda i: (i.Jh, i.Jv))(make_instance(L, 600 + k)), None)[1])
                 for k in range(4)]) / (L * L)
    assert 0.03 < s < 0.15


# ---------------------------------------------------------------------------- Potts q = 3
def py_brute_potts(L, Jh, Jv):
    best, cnt = None, 0
    for cfg in itertools.product(range(3), repeat=L * L):
        t = np.array(cfg).reshape(L, L)
        E = -(Jh * (t[:, :-1] == t[:, 1:])).sum() - (Jv * (t[:-1, :] == t[1:, :])).sum()
        if best is None or E < best:
            best, cnt = E, 1
        elif E == best:
            cnt += 1
    return float(best), cnt


def test_potts_c_brute_equals_python_enumeration():
    for L in (2, 3):
        Jh, Jv, _ = rand_int_instance(L, -2, 2, fields=False)
        assert oracle.brute_potts3(L, Jh, Jv)[:2] == py_brute_potts(L, Jh, Jv)


@pytest.mark.parametrize("L", [1, 2, 3])
def test_potts_dp_equals_brute(L):
    for rep in range(5):
        inst = make_instance(L, 5000 + 10 * L + rep, "pmj", q=3)
        Eb, gb, _ = oracle.brute_potts3(L, inst.Jh, inst.Jv)
        Ed, gd, col = oracle.dp_potts3(L, inst.Jh, inst.Jv, config=True)
        assert (Ed, gd) == (Eb, gb)
        assert oracle.potts3_energy(L, inst.Jh, inst.Jv, col) == Eb
        Jh, Jv, _ = rand_int_instance(L, -2, 3, fields=False)
        assert oracle.dp_potts3(L, Jh, Jv)[:2] == oracle.brute_potts3(L, Jh, Jv)[:2]


def test_potts_dp_equals_brute_L4():
    inst = make_instance(4, 5044, "pmj", q=3)
    assert oracle.dp_potts3(4, inst.Jh, inst.Jv)[:2] == oracle.brute_potts3(4, inst.Jh, inst.Jv)[:2]


def n_proper_3_colourings(L):
    """Independent row-colouring transfer matrix (plain integer arithmetic)."""
    rows = [r for r in itertools.product(range(3), repeat=L)
            if all(r[i] != r[i + 1] for i in range(L - 1))]
    vec = {r: 1 for r in rows}
    for _ in range(L - 1):
        new = {}
        for r2 in rows:
            new[r2] = sum(v for r1, v in vec.items() if all(a != b for a, b in zip(r1, r2)))
        vec = new
    return sum(vec.values())


def test_potts_ferro_and_antiferro_closed_forms():
    golden = [int(x) for x in open(__file__.rsplit("/", 1)[0] + "/golden/grid_3colourings.txt")
              .read().split("\n") if x and not x.startswith("#")]
    for L in range(1, 8):
        Jh = np.ones((L, max(L - 1, 0))); Jv = np.ones((max(L - 1, 0), L))
        E0, g, _ = oracle.dp_potts3(L, Jh, Jv)
        assert E0 == -2 * L * (L - 1) and g == 3
        E0, g, _ = oracle.dp_potts3(L, -Jh, -Jv)
        assert E0 == 0.0 and np.copysign(1.0, E0) == 1.0
        assert g == golden[L - 1]
        if L <= 6:
            assert g == n_proper_3_colourings(L)


def test_potts_symmetries():
    L = 7
    inst = make_instance(L, 5777, "pmj", q=3)
    Jh, Jv = inst.Jh.astype(np.float64), inst.Jv.astype(np.float64)
    E0, g, col = oracle.dp_potts3(L, Jh, Jv, config=True)
    assert g % 3 == 0                       # cyclic colour shift has no fixed point
    assert oracle.potts3_energy(L, Jh, Jv, col) == E0
    assert oracle.dp_potts3(L, Jv.T.copy(), Jh.T.copy())[:2] == (E0, g)
    assert oracle.dp_potts3(L, Jh[:, ::-1].copy(), Jv[:, ::-1].copy())[:2] == (E0, g)
    assert oracle.dp_potts3(L, Jh[::-1, :].copy(), Jv[::-1, :].copy())[:2] == (E0, g)
    assert oracle.dp_potts3(L, 4 * Jh, 4 * Jv)[:2] == (4 * E0, g)


def test_potts_paper_hamiltonian_relation():
    # App. C writes H = sum J M_{s_i s_j}, M = 1 on the diagonal, -1/2 off.
    # H_paper(-J) = 1.5 E_cfg(J) + 0.5 sum_bonds J, same degeneracy.  Check by
    # brute force of the paper's form in Python at L = 2, 3.
    for L in (2, 3):
        Jh, Jv, _ = rand_int_instance(L, -2, 2, fields=False)
        best, cnt = None, 0
        for cfg in itertools.product(range(3), repeat=L * L):
            t = np.array(cfg).reshape(L, L)
            M = lambda a, b: np.where(a == b, 1.0, -0.5)
            H = ((-Jh) * M(t[:, :-1], t[:, 1:])).sum() + ((-Jv) * M(t[:-1, :], t[1:, :])).sum()
            if best is None or H < best - 1e-12:
                best, cnt = H, 1
            elif abs(H - best) <= 1e-12:
                cnt += 1
        E0, g, _ = oracle.dp_potts3(L, Jh, Jv)
        assert abs(best - (1.5 * E0 + 0.5 * (Jh.sum() + Jv.sum()))) < 1e-9 and cnt == g
