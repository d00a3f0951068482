"""Writes tests/golden/config_goldens.json: exact (energy, count) of the BASELINE.json configs at FULL size,
computed by the oracle alone (oracle.frontier_dp, the tree-free transfer-matrix method; SURVEY.md 8(c) Oracle-3).

    python tests/golden/make_config_goldens.py [out.json] [--missing-only]   # minutes of CPU (OpenMP over the host cores)

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
    # the paper's own spin-glass setting (+-J with field 0.5), in integers: J -> 2J, h -> 1, half units
    ("paper-E1 ising 16x16 seed 1 h=0.5 (2J, h=1, half units)", lambda: I.ising_lattice_2d_half_field(16, 16, 1)),
    ("paper-E1 ising 20x20 seed 1 h=0.5 (2J, h=1, half units)", lambda: I.ising_lattice_2d_half_field(20, 20, 1)),
    ("paper-E1 ising 24x24 seed 1 h=0.5 (2J, h=1, half units)", lambda: I.ising_lattice_2d_half_field(24, 24, 1)),
]
# King's subgraphs whose dense frontier table would not fit: oracle.frontier_dp_mis_sparse (independent
# frontier states only); 28x28 6 s, 32x32 ~1.5 min, 36x36 ~8 min, 40x40 longer (one core each)
SPARSE_CASES = [
    ("config5-shape king 28x28 p0.8 seed 1", lambda: I.kings_subgraph(28, 28, 0.8, 1)),
    ("config5-shape king 32x32 p0.8 seed 1", lambda: I.kings_subgraph(32, 32, 0.8, 1)),
    ("config5-shape king 32x32 p0.8 seed 2", lambda: I.kings_subgraph(32, 32, 0.8, 2)),
    ("config5-shape king 36x36 p0.8 seed 1", lambda: I.kings_subgraph(36, 36, 0.8, 1)),
    ("config5 king 40x40 p0.8 seed 1", lambda: I.kings_subgraph(40, 40, 0.8, 1)),
    # more instances of the same ensemble (PAPER.md:95 averages over 10 instances per N)
    ("config5-shape king 36x36 p0.8 seed 2", lambda: I.kings_subgraph(36, 36, 0.8, 2)),
    ("config5-shape king 36x36 p0.8 seed 3", lambda: I.kings_subgraph(36, 36, 0.8, 3)),
    ("config5 king 40x40 p0.8 seed 2", lambda: I.kings_subgraph(40, 40, 0.8, 2)),
    ("config5 king 40x40 p0.8 seed 3", lambda: I.kings_subgraph(40, 40, 0.8, 3)),
]


def main():
    oracle.build()
    out = {"_about": "exact results of oracle.frontier_dp (King's subgraphs of 28x28 and more: oracle.frontier_dp_mis_sparse) on the seeded full-size instances; written by "
                     "tests/golden/make_config_goldens.py (calls only oracle/). energy: Ising min H (Eq. 1, PAPER.md:47), "
                     "MIS max set size (PAPER.md:55); count as a decimal string (may exceed 2^64).", "cases": {}}
    dst = [a for a in sys.argv[1:] if not a.startswith("--")]
    dst = dst[0] if dst else os.path.join(os.path.dirname(os.path.abspath(__file__)), "config_goldens.json")
    if "--missing-only" in sys.argv and os.path.exists(dst):      # keep what is there, add the cases not yet in the file
        with open(dst) as f:
            out["cases"] = json.load(f)["cases"]
    todo = [(n, m, oracle.frontier_dp) for n, m in CASES] + [(n, m, oracle.frontier_dp_mis_sparse) for n, m in SPARSE_CASES]
    for name, make, method in todo:
        if name in out["cases"]:
            continue
        inst = make()
        t0 = time.perf_counter()
        e, c = method(inst)[:2]
        dt = time.perf_counter() - t0
        out["cases"][name] = {"energy": int(e), "count": str(int(c)), "n_vertices": int(inst.n_vertices),
                              "n_edges": int(inst.n_edges), "oracle_seconds": round(dt, 2)}
        print(name, e, c, f"{dt:.1f}s", flush=True)
        with open(dst, "w") as f:                                   # after every case: the long ones can be interrupted
            json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
