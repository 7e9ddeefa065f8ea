"""Host logic: the pass schedule (csrc/planner.h, dumped by ttn_plan_describe) is replayed
(1) against an independent statement of the dependency rule of SURVEY.md 8a-S8
    (derived from PAPER.md:118 "order ... can be arbitrary" + non-commutation of a gate with
    anything that reads its digit), and
(2) numerically, op by op in numpy (float64 + integer counts), against the CPU oracle.
No GPU is needed: this checks what the kernels are told to do, not the kernels.
"""
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
import paper_2008_06888_b200 as ttn
from ttn_inputs import make_instance

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def describe(q, L, call, tmax=None, ride=None, fused=False, nomerge=False):
    """Run ttn_plan_describe in a subprocess so the debug tile overrides can be set."""
    env = dict(os.environ)
    env["TTN_DEBUG_FUSED"] = "1" if fused else "0"
    if nomerge:
        env["TTN_DEBUG_NOMERGE"] = "1"
    if tmax is not None:
        env["TTN_DEBUG_TMAX"] = str(tmax)
    if ride is not None:
        env["TTN_DEBUG_RIDE"] = str(ride)
    code = ("import paper_2008_06888_b200 as t, sys; "
            f"sys.stdout.write(t.plan_describe({q}, {L}, {call}))")
    return subprocess.check_output([sys.executable, "-c", code], cwd=ROOT, env=env, text=True)


def parse(txt):
    head, passes = None, []
    for line in txt.splitlines():
        w = line.split()
        if w[0] == "plan":
            head = dict(kv.split("=") for kv in w[1:])
        elif w[0] == "pass":
            d = {k: int(v) for k, v in (kv.split("=") for kv in w[2:])}
            d["ops"] = []
            passes.append(d)
        elif w[0] == "op":
            d = {k: int(v) for k, v in (kv.split("=") for kv in w[2:])}
            d["type"] = w[1]
            passes[-1]["ops"].append(d)
    return head, passes


VCOL = 255      # csrc/planner.h: the virtual column 0 of a Z3-reduced Potts plan


def validate(q, L, passes, fields, row_aligned, vcol=False):
    """Diagonal frame: only gates are scheduled; g(r,c) needs g(r-1,c-1), g(r-1,c), g(r-1,c+1).
    vcol (Z3-reduced Potts plan): the tiles hold the L - 1 stored digits (digit d = column d + 1); the
    gate on column 0 is an op with c = pos = VCOL and may appear in any pass."""
    g = np.zeros((L, L), dtype=int); g[0, :] = 1          # row 0 needs no gate
    rows_done = 0
    Ld = L - 1 if vcol else L
    for i, ps in enumerate(passes):
        lo, a, b = ps["lo"], ps["a"], ps["b"]
        assert 0 <= lo <= a <= b <= Ld
        tile = list(range(lo)) + list(range(a, b))
        assert len(tile) == len(set(tile)) and len(tile) >= 1
        assert (ps["flags"] & 1) == (1 if i == 0 else 0)          # INIT only on the first pass
        for op in ps["ops"]:
            r, c = op["r"], op["c"]
            assert op["type"] == "g"                               # no diagonal op is ever scheduled
            if vcol and c == VCOL:
                assert op["pos"] == VCOL
                c = 0
            else:
                assert c in tile and tile.index(c) == op["pos"]
                c = c + 1 if vcol else c
            assert 1 <= r < L and g[r, c] == 0 and g[r - 1, c] == 1
            if c > 0: assert g[r - 1, c - 1] == 1
            if c < L - 1: assert g[r - 1, c + 1] == 1
            # the neighbours may be at most one row ahead (same-row gates commute)
            if c > 0 and r + 1 < L: assert g[r + 1, c - 1] == 0
            if c < L - 1 and r + 1 < L: assert g[r + 1, c + 1] == 0
            g[r, c] = 1
        if row_aligned:
            if rows_done < L and g[rows_done].all():
                assert ps["dst"] == rows_done
                rows_done += 1
            else:
                assert ps["dst"] == -1
            if i > 0:
                assert ps["src"] == passes[i - 1]["dst"]
    assert g.all()
    if row_aligned:
        assert rows_done == L
    else:
        assert passes[-1]["flags"] & 2 and all(not (p["flags"] & 2) for p in passes[:-1])


@pytest.mark.parametrize("q,L,call", [(2, 32, 0), (2, 24, 1), (2, 16, 2), (3, 18, 1), (3, 18, 0),
                                      (2, 4, 1), (2, 1, 0), (2, 28, 0), (2, 30, 0), (2, 20, 2),
                                      (3, 12, 0), (2, 34, 0), (2, 15, 0), (2, 14, 1)])
def test_schedule_obeys_dependency_rule(q, L, call):
    head, passes = parse(describe(q, L, call))
    vcol = int(head.get("vcol", 0)) == 1
    assert int(head["L"]) == (L - 1 if vcol else L) and int(head["q"]) == q
    assert vcol == (q == 3 and L >= 10)                   # Potts sweeps beyond one tile run Z3-reduced
    validate(q, L, passes, fields=(q == 2), row_aligned=(call == 2), vcol=vcol)


@pytest.mark.parametrize("L,call,tmax,ride", [(18, 1, None, None), (18, 0, None, None), (12, 0, None, None),
                                              (6, 1, 4, 1), (5, 1, 3, 0), (3, 1, None, None)])
def test_potts_gate_blocks(L, call, tmax, ride):
    """csrc/planner.h mark_gate_blocks (ttn_potts.cuh): the gates of a q = 3 pass are applied in
    blocks of up to three; a block is led by a gate with nb >= 1 and followed by nb - 1 gates with
    nb = 0 on the next columns / tile positions of the SAME row and the SAME round (so they commute,
    PAPER.md:118, and share one conjugation A_{r-1})."""
    _, passes = parse(describe(3, L, call, tmax=tmax, ride=ride))
    sizes = []
    for ps in passes:
        ops = ps["ops"]
        k = 0
        while k < len(ops):
            nb = ops[k]["nb"]
            assert 1 <= nb <= 3 and k + nb <= len(ops)
            for j in range(1, nb):
                o, pr = ops[k + j], ops[k + j - 1]
                assert o["nb"] == 0 and o["first"] == 0
                assert o["r"] == pr["r"] and o["c"] == pr["c"] + 1 and o["pos"] == pr["pos"] + 1
                assert o["c"] != VCOL and pr["c"] != VCOL        # the column-0 gate is a block of its own
            sizes.append(nb)
            k += nb
    assert sum(sizes) == L * (L - 1)
    if L >= 12:
        assert sizes.count(1) < len(sizes) // 2          # most gates ride in blocks of 2 or 3


def test_fusion_cuts_hbm_passes():
    # cross-row fusion brings L=32 from 3 passes per row (93) to ~0.5 per row
    _, passes = parse(describe(2, 32, 0))
    assert len(passes) <= 18
    _, passes = parse(describe(2, 24, 1))
    assert len(passes) <= 12
    head, fpasses = parse_fused(describe(2, 32, 0, fused=True))
    assert len(fpasses) <= 24
    # q = 3: beam search over tile sequences (planner.h make_plan_beam) vs the cyclic tile order
    # (Z3-reduced: passes over a third of the state)
    _, passes = parse(describe(3, 18, 1))
    assert len(passes) <= 15
    _, passes = parse(describe(3, 18, 0))
    assert len(passes) <= 11


# ------------------------------------------------------------------ fused register-phase schedule
# Diagonal frame (csrc/planner.h): the row diagonals are folded into the gates by conjugating
# every gate with the accumulated diagonal operator, G''_r(c) = A_{r-1}^{-1} G_r(c) A_{r-1}.
# Restated here independently: with H_c, K_c the sums of h[r'][c], Jh[r'][c] over r' < r,
#     a' = max(a, b + m - 2 rho), b' = max(b, a + m + 2 rho),  m = -2 Jv[r-1][c],
#     rho = H_c + K_{c-1} sigma_{c-1} + K_c sigma_{c+1};   result = max_s(V(s) + A_{L-1}(s)).
# Dependency rule in this frame: g(r,c) after g(r-1,c-1), g(r-1,c), g(r-1,c+1).
# register-index bit -> tile digit, as documented in csrc/planner.h (fused_digit_of_bit)
# (mirrored layouts: layout B holds the register digits in reverse chain order)
DIGIT_OF_BIT = {(1, 0): [5, 6, 0, 1, 2, 3, 4], (1, 1): [6, 5, 11, 10, 9, 8, 7],
                (0, 0): [4, 5, 6, 0, 1, 2, 3], (0, 1): [4, 3, 2, 8, 7, 6, 5]}


def parse_fused(txt):
    head, passes = None, []
    for line in txt.splitlines():
        w = line.split()
        if w[0] == "fused":
            head = dict(kv.split("=") for kv in w[1:])
        elif w[0] == "fpass":
            d = {k: int(v) for k, v in (kv.split("=") for kv in w[2:])}
            d["mops"] = []
            passes.append(d)
        elif w[0] == "m":
            d = {"code": w[1]}
            d.update({k: int(v) for k, v in (kv.split("=") for kv in w[2:])})
            d["gates"] = []
            passes[-1]["mops"].append(d)
        elif w[0] == "g":
            passes[-1]["mops"][-1]["gates"].append({k: int(v) for k, v in (kv.split("=") for kv in w[1:])})
    return head, passes


# counting geometry (csrc/planner.h GEOM_COUNT): 5 register digits, bit i = chain position i
DIGIT_OF_BIT_COUNT = {(1, 0): [0, 1, 2, 3, 4], (1, 1): [9, 8, 7, 6, 5],
                      (0, 0): [0, 1, 2, 3, 4], (0, 1): [6, 5, 4, 3, 2]}


# Tropical<i16> geometry (GEOM_I16): column 0 is the half of a 32-bit word (pseudo register bit 7
# of the LOW tile), column c >= 1 is word digit c - 1 with the f32 maps
DIGIT_OF_BIT_I16 = {(1, 0): [1 + d for d in [5, 6, 0, 1, 2, 3, 4]] + [0], (1, 1): [1 + d for d in [6, 5, 11, 10, 9, 8, 7]] + [0],
                    (0, 0): [4, 5, 6, 0, 1, 2, 3], (0, 1): [4, 3, 2, 8, 7, 6, 5]}


# flip-reduced f32 geometry (GEOM_F32_Z2, h = 0): column 0 is not stored (the half-state holds the
# configurations with column 0 up); column c >= 1 is digit c - 1 with the f32 maps; the gate on
# column 0 ("flip gate", k = -1) may end any round of a LOW pass
DIGIT_OF_BIT_Z2 = {(1, 0): [1 + d for d in [5, 6, 0, 1, 2, 3, 4]], (1, 1): [1 + d for d in [6, 5, 11, 10, 9, 8, 7]],
                   (0, 0): [4, 5, 6, 0, 1, 2, 3], (0, 1): [4, 3, 2, 8, 7, 6, 5]}


# flip-reduced counting geometry (GEOM_COUNT_Z2): column c >= 1 is digit c - 1 with the counting maps
DIGIT_OF_BIT_COUNT_Z2 = {(1, 0): [1, 2, 3, 4, 5], (1, 1): [10, 9, 8, 7, 6],
                         (0, 0): [0, 1, 2, 3, 4], (0, 1): [6, 5, 4, 3, 2]}


# flip-reduced Tropical<i16> geometry (GEOM_I16_Z2): column 1 is the half of a word (pseudo bit 7),
# column c >= 2 is word digit c - 2
DIGIT_OF_BIT_I16_Z2 = {(1, 0): [2 + d for d in [5, 6, 0, 1, 2, 3, 4]] + [1], (1, 1): [2 + d for d in [6, 5, 11, 10, 9, 8, 7]] + [1],
                       (0, 0): [4, 5, 6, 0, 1, 2, 3], (0, 1): [4, 3, 2, 8, 7, 6, 5]}


def fused_to_gates(L, fpasses, count=False, i16=False, config=False, z2=False):
    """Check the structure of the micro-op program (layouts, register bits, rounds) and the
    three-point-stencil dependency rule; return the flat (r, c) gate sequence."""
    flat = []
    grow = [1] * L                                   # rows complete per digit (row 0 needs no gate)
    for i, ps in enumerate(fpasses):
        a, Wt, low = ps["a"], ps["W"], ps["low"]
        wl, wh, rb = ((11, 7, 5) if z2 else (10, 7, 5)) if count else ((14 if z2 else 13, 9, 8 if low else 7) if i16 else ((13, 9, 7) if z2 else (12, 9, 7)))
        dmap = (DIGIT_OF_BIT_COUNT_Z2 if z2 else DIGIT_OF_BIT_COUNT) if count else \
               ((DIGIT_OF_BIT_I16_Z2 if z2 else DIGIT_OF_BIT_I16) if i16 else (DIGIT_OF_BIT_Z2 if z2 else DIGIT_OF_BIT))
        amin = 4 + (1 if i16 else 0) + (1 if z2 else 0)
        assert (low == 1 and a == 0 and Wt == wl) or (low == 0 and a >= amin and Wt == wh)
        assert a + Wt <= L
        assert (ps["flags"] & 1) == (1 if i == 0 else 0)
        last = i == len(fpasses) - 1 and not config
        assert bool(ps["flags"] & 2) == last
        if low:
            assert ps["first"] == 1 and ps["last"] == 1     # coalesced global layout
        layout = ps["first"]
        assert ps["mops"][-1]["code"] == ("final" if last else "end")
        assert len(ps["mops"]) <= 128
        ngates = 0
        for m in ps["mops"][:-1]:
            code = m["code"]
            if code == "ckpt":
                assert config and ps["ckpt"] >= 1 and (not low or layout == 1)
                assert all(g >= ps["ckpt"] + 1 for g in grow)             # the row is complete where it is stored
                assert all(g <= ps["ckpt"] + 1 for g in grow)             # ... and nothing of the next row is in it
                continue
            if code == "xAB":
                assert layout == 0
                layout = 1
            elif code == "xBA":
                assert layout == 1
                layout = 0
            else:
                flip = m.get("flip", 0)
                assert not flip or (z2 and low)                      # flip gates: LOW passes of Z2 plans only
                assert code == "round" and (flip or 0 < m["mask"]) and m["mask"] < (1 << rb) and m["first"] == ngates
                bits = [k for k in range(rb) if m["mask"] >> k & 1] + ([-1] if flip else [])
                assert [g["k"] for g in m["gates"]] == bits          # ascending register bits, the flip gate last
                before = list(grow)
                for g in m["gates"]:
                    c, r = g["c"], g["r"]
                    if g["k"] < 0:
                        assert c == 0
                    else:
                        assert c == a + dmap[(low, layout)][g["k"]]  # register bit <-> column
                        assert not z2 or c >= 1
                    assert g["layout"] == layout
                    # legal at the START of the round: every gate of a round commutes with the others
                    assert 1 <= r < L and before[c] == r
                    assert c == 0 or before[c - 1] >= r
                    assert c == L - 1 or before[c + 1] >= r
                    grow[c] += 1
                    flat.append((r, c))
                ngates += len(bits)
        assert layout == ps["last"] and ngates == ps["gates"] <= 160
    assert grow == [L] * L
    return flat


@pytest.mark.parametrize("L", [12, 13, 14, 16, 17, 20, 24, 28, 32, 34])
def test_fused_schedule_obeys_dependency_rule(L):
    head, fpasses = parse_fused(describe(2, L, 0, fused=True))
    assert int(head["L"]) == L
    flat = fused_to_gates(L, fpasses)
    assert len(flat) == L * (L - 1) == len(set(flat))


def replay_diagonal_frame(L, gates, Jh, Jv, h):
    """numpy float64 replay of the conjugated gates in schedule order (Ising, energy only)."""
    N = 2 ** L
    s = np.arange(N)
    sig = [1 - 2 * ((s >> c) & 1) for c in range(L)]
    Hacc = np.cumsum(h, axis=0) if h is not None else np.zeros((L, L))
    Kacc = np.cumsum(Jh, axis=0)
    V = np.zeros(N)
    defer = 0.0
    for (r, c) in gates:
        J = Jv[r - 1, c]
        defer += J
        rho = Hacc[r - 1, c] * np.ones(N)
        if c > 0:
            rho = rho + Kacc[r - 1, c - 1] * sig[c - 1]
        if c < L - 1:
            rho = rho + Kacc[r - 1, c] * sig[c + 1]
        ia = s[(s >> c) & 1 == 0]
        ib = ia | (1 << c)
        xa, xb = V[ia].copy(), V[ib].copy()
        V[ia] = np.maximum(xa, xb - 2 * J - 2 * rho[ia])
        V[ib] = np.maximum(xb, xa - 2 * J + 2 * rho[ia])
    A = np.zeros(N)
    for c in range(L):
        A += Hacc[L - 1, c] * sig[c]
        if c < L - 1:
            A += Kacc[L - 1, c] * sig[c] * sig[c + 1]
    m = (V + A).max() + defer
    return 0.0 if m == 0 else -m


@pytest.mark.parametrize("L", [10, 11, 12, 14, 17, 20, 24, 28, 32])
def test_fused_count_schedule_obeys_dependency_rule(L):
    head, fpasses = parse_fused(describe(2, L, 1, fused=True))
    assert int(head["L"]) == L
    flat = fused_to_gates(L, fpasses, count=True)
    assert len(flat) == L * (L - 1) == len(set(flat))


@pytest.mark.parametrize("L", [13, 14, 15, 18, 22, 24, 28, 32, 34])
def test_fused_i16_schedule_obeys_dependency_rule(L):
    head, fpasses = parse_fused(describe(2, L, 3, fused=True))
    assert int(head["L"]) == L
    flat = fused_to_gates(L, fpasses, i16=True)
    assert len(flat) == L * (L - 1) == len(set(flat))


@pytest.mark.parametrize("L", [14, 15, 16, 19, 23, 24, 28, 30, 32, 34])
def test_fused_z2_schedule_obeys_dependency_rule(L):
    """h = 0 flip reduction: same stencil rule; the gates on column 0 appear as
    flip gates in LOW passes, exactly one per row."""
    head, fpasses = parse_fused(describe(2, L, 4, fused=True))
    assert int(head["L"]) == L
    flat = fused_to_gates(L, fpasses, z2=True)
    assert len(flat) == L * (L - 1) == len(set(flat))
    assert sorted(r for r, c in flat if c == 0) == list(range(1, L))


@pytest.mark.parametrize("L", [12, 13, 14, 17, 20, 24, 28, 32])
def test_fused_count_z2_schedule_obeys_dependency_rule(L):
    head, fpasses = parse_fused(describe(2, L, 5, fused=True))
    assert int(head["L"]) == L
    flat = fused_to_gates(L, fpasses, count=True, z2=True)
    assert len(flat) == L * (L - 1) == len(set(flat))
    assert sorted(r for r, c in flat if c == 0) == list(range(1, L))


@pytest.mark.parametrize("L", [15, 16, 17, 20, 24, 28, 32, 34])
def test_fused_i16_z2_schedule_obeys_dependency_rule(L):
    head, fpasses = parse_fused(describe(2, L, 6, fused=True))
    assert int(head["L"]) == L
    flat = fused_to_gates(L, fpasses, i16=True, z2=True)
    assert len(flat) == L * (L - 1) == len(set(flat))
    assert sorted(r for r, c in flat if c == 0) == list(range(1, L))


def replay_z2_half_state(L, gates, Jh, Jv, count=False):
    """numpy float64 replay of a flip-reduced schedule on the HALF state, restated from the symmetry:
    with h = 0 every intermediate state W of the sweep obeys W[s] = W[~s] (each gate (A2) PAPER.md:242
    and each diagonal (A4) PAPER.md:251 commutes with the global flip of Eq. (1)), so
    only u = (s_1 .. s_{L-1}) with s_0 = 0 (sigma_0 = +1) is stored and the partner of u under the
    column-0 gate, the element with s_0 = 1, is W[~u].  Gates in the diagonal frame as above."""
    N = 2 ** (L - 1)
    u = np.arange(N)
    sig = [np.ones(N)] + [1 - 2 * ((u >> (c - 1)) & 1) for c in range(1, L)]
    Kacc = np.cumsum(Jh, axis=0)
    V = np.zeros(N)
    n = np.ones(N)                       # counts as float64: exact below 2^53 (the sizes replayed here)
    defer = 0.0

    def oplus(xk, nk, xc, nc):           # Eq. (4): keep (+) candidate
        return np.maximum(xk, xc), nk * (xk >= xc) + nc * (xc >= xk)

    for (r, c) in gates:
        J = Jv[r - 1, c]
        defer += J
        rho = np.zeros(N)
        if c > 0:
            rho = rho + Kacc[r - 1, c - 1] * sig[c - 1]
        if c < L - 1:
            rho = rho + Kacc[r - 1, c] * sig[c + 1]
        if c == 0:
            co = (N - 1) ^ u                                          # a' = a (+) (b + m - 2 rho), b = W[~u]
            V, n = oplus(V, n, V[co] - 2 * J - 2 * rho, n[co])
        else:
            ia = u[(u >> (c - 1)) & 1 == 0]
            ib = ia | (1 << (c - 1))
            xa, xb, na, nb = V[ia].copy(), V[ib].copy(), n[ia].copy(), n[ib].copy()
            V[ia], n[ia] = oplus(xa, na, xb - 2 * J - 2 * rho[ia], nb)
            V[ib], n[ib] = oplus(xb, nb, xa - 2 * J + 2 * rho[ia], na)
    A = np.zeros(N)
    for c in range(L - 1):
        A += Kacc[L - 1, c] * sig[c] * sig[c + 1]
    x = V + A
    m = x.max()
    E0 = 0.0 if m + defer == 0 else -(m + defer)
    if count:
        return E0, 2 * int(n[x == m].sum())       # the stored half holds one of every flip pair
    return E0


@pytest.mark.parametrize("L", [14, 15, 17])
def test_fused_z2_schedule_replay_matches_oracle(L):
    _, fpasses = parse_fused(describe(2, L, 4, fused=True))
    flat = fused_to_gates(L, fpasses, z2=True)
    rng = np.random.default_rng(200 + L)
    Jh = rng.integers(-2, 3, size=(L, L - 1)).astype(float)
    Jv = rng.integers(-2, 3, size=(L - 1, L)).astype(float)
    Eo, _, _ = oracle.dp_ising(L, Jh, Jv, None, count=False)
    assert replay_z2_half_state(L, flat, Jh, Jv) == Eo
    Jh, Jv = rng.normal(size=Jh.shape), rng.normal(size=Jv.shape)
    Eo, _, _ = oracle.dp_ising(L, Jh, Jv, None, count=False)
    assert abs(replay_z2_half_state(L, flat, Jh, Jv) - Eo) <= 1e-9 * abs(Eo)


@pytest.mark.parametrize("L", [12, 13, 15])
def test_fused_count_z2_schedule_replay_matches_oracle(L):
    _, fpasses = parse_fused(describe(2, L, 5, fused=True))
    flat = fused_to_gates(L, fpasses, count=True, z2=True)
    rng = np.random.default_rng(300 + L)
    for trial in range(2):
        Jh = rng.integers(-1, 2, size=(L, L - 1)).astype(float)       # many ties
        Jv = rng.integers(-1, 2, size=(L - 1, L)).astype(float)
        Eo, go, _ = oracle.dp_ising(L, Jh, Jv, None)
        assert go < 2 ** 53
        assert replay_z2_half_state(L, flat, Jh, Jv, count=True) == (Eo, go)


def test_z2_describe_falls_back_below_two_tiles():
    """L = 13: the half-state is a single (self-complementary) LOW tile: the plain schedule runs."""
    assert describe(2, 13, 4, fused=True) == describe(2, 13, 0, fused=True)
    assert describe(2, 11, 5, fused=True) == describe(2, 11, 1, fused=True)
    assert describe(2, 14, 6, fused=True) == describe(2, 14, 3, fused=True)


@pytest.mark.parametrize("L", [12, 13, 16, 20, 21, 22, 28])
def test_fused_row_aligned_schedule(L):
    """ttn_ground_config on the fused kernel: every row boundary is a checkpoint; the pass that
    completes row r writes C_r, the next one reads it (src/dst chain)."""
    head, fpasses = parse_fused(describe(2, L, 2, fused=True, nomerge=True))
    flat = fused_to_gates(L, fpasses, config=True)
    assert len(flat) == L * (L - 1)
    rows = [r for r, c in flat]
    assert rows == sorted(rows)                              # no gate of row r+1 before row r is complete
    assert fpasses[0]["gates"] == 0 and fpasses[0]["src"] == -1 and fpasses[0]["dst"] == 0
    done, seen = 0, 0
    for i, ps in enumerate(fpasses[1:], 1):
        assert ps["src"] == fpasses[i - 1]["dst"]
        seen += ps["gates"]
        if seen == (done + 1) * L:
            done += 1
            assert ps["dst"] == done
        else:
            assert ps["dst"] == -1
    assert done == L - 1


@pytest.mark.parametrize("L", [14, 16, 21, 30, 32])
def test_fused_z2_row_aligned_schedule(L):
    """ttn_ground_config with h = 0: the row-aligned plan on the flip-reduced geometry (checkpoints are
    half-states); rows complete in order, one flip gate (column 0) per row, src/dst chain intact."""
    head, fpasses = parse_fused(describe(2, L, 7, fused=True, nomerge=True))
    flat = fused_to_gates(L, fpasses, config=True, z2=True)
    assert len(flat) == L * (L - 1) == len(set(flat))
    rows = [r for r, c in flat]
    assert rows == sorted(rows)
    assert sorted(r for r, c in flat if c == 0) == list(range(1, L))
    assert fpasses[0]["gates"] == 0 and fpasses[0]["src"] == -1 and fpasses[0]["dst"] == 0
    done, seen = 0, 0
    for i, ps in enumerate(fpasses[1:], 1):
        assert ps["src"] == fpasses[i - 1]["dst"]
        seen += ps["gates"]
        if seen == (done + 1) * L:
            done += 1
            assert ps["dst"] == done
        else:
            assert ps["dst"] == -1
    assert done == L - 1


@pytest.mark.parametrize("L,call", [(13, 2), (16, 2), (20, 2), (21, 2)])
def test_fused_merged_row_schedule(L, call):
    """Merged row-aligned plan (low tile + one high tile): the tile order alternates from row to row and the
    two passes on the same tile merge around a mid-pass checkpoint store: L passes; every C_r (0 < r < L-1)
    is written by an MC_CKPT micro-op exactly where row r is complete and row r + 1 untouched (checked
    inside fused_to_gates), C_0 and C_{L-1} by the first and the last pass."""
    z2 = call == 7
    head, fpasses = parse_fused(describe(2, L, call, fused=True))
    flat = fused_to_gates(L, fpasses, config=True, z2=z2)
    assert len(flat) == L * (L - 1) == len(set(flat))
    assert len(fpasses) == L + 1
    assert fpasses[0]["dst"] == 0 and fpasses[1]["src"] == 0 and fpasses[-1]["dst"] == L - 1
    assert [ps["ckpt"] for ps in fpasses[2:-1]] == list(range(1, L - 1))
    assert all(ps["src"] == -1 and ps["dst"] == -1 for ps in fpasses[2:-1])
    assert [ps["low"] for ps in fpasses[1:]] == [(i + 1) % 2 for i in range(L)]     # low, high, low, ...
    for ps in fpasses:
        assert [m["code"] for m in ps["mops"]].count("ckpt") == (1 if ps["ckpt"] >= 0 else 0)


@pytest.mark.parametrize("L", [12, 13, 16])
def test_fused_schedule_replay_matches_oracle(L):
    _, fpasses = parse_fused(describe(2, L, 0, fused=True))
    flat = fused_to_gates(L, fpasses)
    rng = np.random.default_rng(L)
    Jh = rng.integers(-2, 3, size=(L, L - 1)).astype(float)
    Jv = rng.integers(-2, 3, size=(L - 1, L)).astype(float)
    h = rng.integers(-1, 2, size=(L, L)).astype(float)
    Eo, _, _ = oracle.dp_ising(L, Jh, Jv, h, count=False)
    assert replay_diagonal_frame(L, flat, Jh, Jv, h) == Eo
    Jh, Jv, h = rng.normal(size=Jh.shape), rng.normal(size=Jv.shape), rng.normal(size=h.shape)
    Eo, _, _ = oracle.dp_ising(L, Jh, Jv, h, count=False)
    assert abs(replay_diagonal_frame(L, flat, Jh, Jv, h) - Eo) <= 1e-9 * abs(Eo)


# ------------------------------------------------------------------------------- numeric replay
def digits(q, L):
    s = np.arange(q ** L)
    return [(s // q ** c) % q for c in range(L)]


def replay(q, L, passes, Jh, Jv, h):
    """Apply the gate list to the full state in numpy in the diagonal frame, restated here from
    the paper's gates: x float64, n Python-int (object) counts.  With A_{r-1}(s) the sum of all
    diagonal gates (A3), (A4) of rows < r, gate g(r,c) is  G'' = A^-1 G A:
        cand(t -> t') = x[t] + w(t,t') + R(t) - R(t'),   R(t) = the terms of A_{r-1} that contain digit c
    and the result is  (+)_s ( x[s] (.) A_{L-1}(s) )."""
    N = q ** L
    x = np.zeros(N); n = np.ones(N, dtype=object)
    dig = digits(q, L)
    idx = np.arange(N)
    H = np.cumsum(h, axis=0) if h is not None else np.zeros((L, L))
    K = np.cumsum(Jh, axis=0)

    def two(Kc, d0, d1):
        return Kc * (1 - 2 * d0) * (1 - 2 * d1) if q == 2 else Kc * (d0 == d1)

    def R_of(r, c, t, sel):
        out = np.zeros(sel.size)
        if q == 2:
            out = out + H[r - 1, c] * (1 - 2 * t)
        if c > 0:
            out = out + two(K[r - 1, c - 1], dig[c - 1][sel], t)
        if c < L - 1:
            out = out + two(K[r - 1, c], t, dig[c + 1][sel])
        return out

    for ps in passes:
        for op in ps["ops"]:
            assert op["type"] == "g"
            r, c = op["r"], op["c"]
            J = Jv[r - 1, c]
            st = q ** c
            base = idx[dig[c] == 0]
            olds = [(x[base + t * st].copy(), n[base + t * st].copy()) for t in range(q)]
            Rs = [R_of(r, c, t, base) for t in range(q)]
            for tn in range(q):
                bx = None
                for t in range(q):
                    w = J * (1 - 2 * t) * (1 - 2 * tn) if q == 2 else J * (t == tn)
                    cx, cn = olds[t][0] + w + Rs[t] - Rs[tn], olds[t][1]
                    if bx is None:
                        bx, bn = cx.copy(), cn.copy()
                    else:
                        gt, eq = cx > bx, cx == bx
                        bn = np.where(gt, cn, np.where(eq, bn + cn, bn))
                        bx = np.maximum(bx, cx)
                x[base + tn * st] = bx; n[base + tn * st] = bn
    A = np.zeros(N)
    for c in range(L):
        if q == 2:
            A = A + H[L - 1, c] * (1 - 2 * dig[c])
        if c < L - 1:
            A = A + two(K[L - 1, c], dig[c], dig[c + 1])
    x = x + A
    m = x.max()
    return (0.0 if m == 0 else -m), int(sum(n[x == m]))


def replay_z3(L, passes, Jh, Jv):
    """Z3-reduced Potts replay, restated from the symmetry: E = -sum J delta (App. C PAPER.md:296 in
    BASELINE.json's reading) is invariant under t -> t + 1 (mod 3) on every site, so every intermediate
    state W of the sweep obeys W[t] = W[rho t].  Stored: H[rest] = W[0, rest] over the digits of columns
    1 .. L-1.  A gate on column c >= 1 acts inside H (column 1 sees colour 0 on its left).  The gate on
    column 0 acts on x_k = W[k, rest] = H[rho^-k rest] (every digit of rest minus k), k = 0, 1, 2."""
    Ld = L - 1
    N = 3 ** Ld
    x = np.zeros(N); n = np.ones(N, dtype=object)
    idx = np.arange(N)
    dig = [(idx // 3 ** d) % 3 for d in range(Ld)]          # dig[d] = colour of column d + 1
    K = np.cumsum(Jh, axis=0)

    def rot_minus(k):                                       # index of rho^-k rest
        out = np.zeros(N, dtype=np.int64)
        for d in range(Ld):
            out += ((dig[d] - k) % 3) * 3 ** d
        return out

    rm = [idx, rot_minus(1), rot_minus(2)]

    def gate3(olds, J, Rs):
        news = []
        for tn in range(3):
            bx = None
            for t in range(3):
                cx, cn = olds[t][0] + J * (t == tn) + Rs[t] - Rs[tn], olds[t][1]
                if bx is None:
                    bx, bn = cx.copy(), cn.copy()
                else:
                    gt, eq = cx > bx, cx == bx
                    bn = np.where(gt, cn, np.where(eq, bn + cn, bn))
                    bx = np.maximum(bx, cx)
            news.append((bx, bn))
        return news

    for ps in passes:
        for op in ps["ops"]:
            r = op["r"]
            if op["c"] == VCOL:                             # column 0: R(t) = K_0 delta(t, colour of column 1)
                J = Jv[r - 1, 0]
                sel = idx                                   # every rest once, as the k = 0 member
                olds = [(x[rm[k]].copy(), n[rm[k]].copy()) for k in range(3)]
                Rs = [K[r - 1, 0] * (dig[0] == t) for t in range(3)]
                news = gate3(olds, J, Rs)
                x = news[0][0]; n = news[0][1]              # H'[rest] = W'[0, rest]; the others follow by symmetry
                for k in (1, 2):                            # ... and must agree with what the symmetry predicts
                    assert np.array_equal(news[k][0], x[rm[k]])
                continue
            d = op["c"]; c = d + 1
            J = Jv[r - 1, c]
            st = 3 ** d
            base = idx[dig[d] == 0]
            olds = [(x[base + t * st].copy(), n[base + t * st].copy()) for t in range(3)]
            left = dig[d - 1][base] if d > 0 else np.zeros(base.size, dtype=np.int64)     # column 0 = colour 0
            Rs = []
            for t in range(3):
                R = K[r - 1, c - 1] * (left == t)
                if c < L - 1:
                    R = R + K[r - 1, c] * (t == dig[d + 1][base])
                Rs.append(R)
            news = gate3(olds, J, Rs)
            for t in range(3):
                x[base + t * st] = news[t][0]; n[base + t * st] = news[t][1]
    A = K[L - 1, 0] * (dig[0] == 0)
    for d in range(Ld - 1):
        A = A + K[L - 1, d + 1] * (dig[d] == dig[d + 1])
    x = x + A
    m = x.max()
    return (0.0 if m == 0 else -m), 3 * int(sum(n[x == m]))


@pytest.mark.parametrize("q,L,call,tmax,ride", [
    (2, 8, 1, 5, 2), (2, 9, 0, 4, 1), (2, 7, 1, 3, 1), (2, 10, 1, 6, 3), (2, 6, 2, 4, 2),
    (3, 6, 1, 3, 1), (3, 5, 1, 2, 1), (3, 7, 0, 4, 2), (2, 8, 1, 13, 3), (3, 7, 1, 3, 0), (3, 4, 1, 2, 1),
])
def test_schedule_replay_matches_oracle(q, L, call, tmax, ride):
    head, passes = parse(describe(q, L, call, tmax, ride))
    vcol = int(head.get("vcol", 0)) == 1
    validate(q, L, passes, fields=(q == 2), row_aligned=(call == 2), vcol=vcol)
    if tmax < L:
        assert len(passes) > 1
    if vcol:
        assert q == 3
        for seed in range(3):
            inst = make_instance(L, 900 + seed, "pmj", q=3)
            assert replay_z3(L, passes, inst.Jh, inst.Jv) == oracle.dp_potts3(L, inst.Jh, inst.Jv)[:2]
        rng = np.random.default_rng(L)
        Jh = rng.integers(-2, 3, size=(L, L - 1)).astype(float)
        Jv = rng.integers(-2, 3, size=(L - 1, L)).astype(float)
        assert replay_z3(L, passes, Jh, Jv) == oracle.dp_potts3(L, Jh, Jv)[:2]
        return
    for seed in range(3):
        if q == 2:
            rng = np.random.default_rng(seed)
            Jh = rng.integers(-2, 3, size=(L, L - 1)).astype(float)
            Jv = rng.integers(-2, 3, size=(L - 1, L)).astype(float)
            h = rng.integers(-1, 2, size=(L, L)).astype(float)
            E0, g = replay(q, L, passes, Jh, Jv, h)
            Eo, go, _ = oracle.dp_ising(L, Jh, Jv, h)
        else:
            inst = make_instance(L, 900 + seed, "pmj", q=3)
            E0, g = replay(q, L, passes, inst.Jh, inst.Jv, None)
            Eo, go, _ = oracle.dp_potts3(L, inst.Jh, inst.Jv)
        assert (E0, g) == (Eo, go)
