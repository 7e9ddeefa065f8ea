"""CPU oracle for the tropical tensor-network sweep -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2008_06888_b200`` (the CUDA path) and neither imports the other.
See ``ttn_oracle.c`` for what is computed and which PAPER.md passages it follows.
"""
from .ttn_oracle import (  # noqa: F401
    build,
    brute_ising,
    brute_potts3,
    dp_ising,
    dp_potts3,
    ising_energy,
    potts3_energy,
    num_threads,
    OracleOverflow,
)
