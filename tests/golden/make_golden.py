"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ (the CPU
oracle) on instances from ttn_inputs (the seeded generator).  Nothing here touches the CUDA
path.  Usage:

    python tests/golden/make_golden.py ising_count 24 3000 3016     # cfg 3 (16 seeds)
    python tests/golden/make_golden.py ising_energy 32 4000 4001    # cfg 4 (34 GB, ~hours)
    python tests/golden/make_golden.py potts_count 18 5000 5004     # cfg 5
    python tests/golden/make_golden.py ising_gauss 16 2000 2256     # cfg 2 (E0 + sigma energy)
    python tests/golden/make_golden.py chimera 6 7006 7007          # chimera graph, 6 x 6 cells (L = M = N), dp_chimera

Each run appends/updates lines "kind L seed E0 g" in tests/golden/oracle_values.txt (g = -1
when not computed; E0 printed with repr() so float64 round-trips exactly).
"""
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from ttn_inputs import make_instance  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_values.txt")
HEADER = (
    "# kind L seed E0 g  -- written by tests/golden/make_golden.py from oracle/ (O-dp) on\n"
    "# ttn_inputs.make_instance(L, seed, ...).  kinds: ising_count/ising_energy = +-J h=0 (cfg 3/4\n"
    "# distribution), potts_count = +-J 3-state Potts (cfg 5), ising_gauss = Gaussian J,h (cfg 2),\n"
    "# chimera = +-J chimera graph of L x L unit cells, ttn_inputs.make_chimera_instance(L, L, seed), oracle.chimera_oracle.dp_chimera.\n"
)


def load():
    rows = {}
    if os.path.exists(OUT):
        for line in open(OUT):
            if line.startswith("#") or not line.strip():
                continue
            k, L, seed, E0, g = line.split()
            rows[(k, int(L), int(seed))] = (E0, g)
    return rows


def save(rows):
    with open(OUT + ".tmp", "w") as f:
        f.write(HEADER)
        for (k, L, seed) in sorted(rows):
            E0, g = rows[(k, L, seed)]
            f.write(f"{k} {L} {seed} {E0} {g}\n")
    os.replace(OUT + ".tmp", OUT)


def main():
    kind, L, s0, s1 = sys.argv[1], int(sys.argv[2]), int(sys.argv[3]), int(sys.argv[4])
    for seed in range(s0, s1):
        t = time.time()
        if kind == "ising_count":
            i = make_instance(L, seed, "pmj")
            E0, g, _ = oracle.dp_ising(L, i.Jh, i.Jv, None, count=True)
        elif kind == "ising_energy":
            i = make_instance(L, seed, "pmj")
            E0, g, _ = oracle.dp_ising(L, i.Jh, i.Jv, None, count=False)
            g = -1
        elif kind == "potts_count":
            i = make_instance(L, seed, "pmj", q=3)
            E0, g, _ = oracle.dp_potts3(L, i.Jh, i.Jv, count=True)
        elif kind == "ising_gauss":
            i = make_instance(L, seed, "gauss", fields=True)
            E0, g, _ = oracle.dp_ising(L, i.Jh, i.Jv, i.h, count=False)
            g = -1
        elif kind == "chimera":
            from oracle import chimera_oracle
            from ttn_inputs import make_chimera_instance
            i = make_chimera_instance(L, L, seed)
            E0, g = chimera_oracle.dp_chimera(L, L, 4, i.K, i.Jv, i.Jh)
        else:
            raise SystemExit("unknown kind")
        rows = load()
        rows[(kind, L, seed)] = (repr(float(E0)), str(g))
        save(rows)
        print(f"{kind} L={L} seed={seed} E0={E0!r} g={g} ({time.time() - t:.1f}s)", flush=True)


if __name__ == "__main__":
    main()
