"""Writes tests/golden/config_goldens.json: exact (energy, count) of the BASELINE.json configs at FULL size,
computed by the oracle alone (oracle.frontier_dp, the tree-free transfer-matrix method; SURVEY.md 8(c) Oracle-3).

    python tests/golden/make_config_goldens.py [out.json]   # minutes of CPU (OpenMP over the host cores)

Nothing here touches the CUDA path: the GPU parity tests read the file this script writes.
Instances come from the seeded generators (paper_2602_05470_b200/instances.py holds no arithmetic of the method).
"""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from paper_2602_05470_b200 import instances as I  # noqa: E402

CASES = [
    ("config1 ising 6x6 seed 1", lambda: I.ising_lattice_2d(6, 6, 1)),
    ("config1 ising 6x6 seed 2", lambda: I.ising_lattice_2d(6, 6, 2)),
    ("config2 king 12x12 p0.8 seed 1", lambda: I.kings_subgraph(12, 12, 0.8, 1)),
    ("config3 ising 24x24 seed 1", lambda: I.ising_lattice_2d(24, 24, 1)),
    ("config4b ising 5x5x5 seed 1", lambda: I.ising_lattice_3d(5, 5, 5, 1)),
    ("config5-shape king 16x16 p0.8 seed 1", lambda: I.kings_subgraph(16, 16, 0.8, 1)),
    ("config5-shape king 20x20 p0.8 seed 1", lambda: I.kings_subgraph(20, 20, 0.8, 1)),
    ("config5-shape king 24x24 p0.8 seed 1", lambda: I.kings_subgraph(24, 24, 0.8, 1)),
]


def main():
    oracle.build()
    out = {"_about": "exact results of oracle.frontier_dp on the seeded full-size instances; written by "
                     "tests/golden/make_config_goldens.py (calls only oracle/). energy: Ising min H (Eq. 1, PAPER.md:47), "
                     "MIS max set size (PAPER.md:55); count as a decimal string (may exceed 2^64).", "cases": {}}
    for name, make in CASES:
        inst = make()
        t0 = time.perf_counter()
        e, c = oracle.frontier_dp(inst)[:2]
        dt = time.perf_counter() - t0
        out["cases"][name] = {"energy": int(e), "count": str(int(c)), "n_vertices": int(inst.n_vertices),
                              "n_edges": int(inst.n_edges), "oracle_seconds": round(dt, 2)}
        print(name, e, c, f"{dt:.1f}s", flush=True)
    dst = sys.argv[1] if len(sys.argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)), "config_goldens.json")
    with open(dst, "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
