"""time-to-exact (E0, count) on the BASELINE.json lattice configurations, through the C ABI only.

    python -m paper_2602_05470_b200.time_to_solve [--configs 1 2 3 4b 5] [--king-sizes 16 20 24 28] [--repeat 5]

Prints one JSON line per solve: instance, fixed set / batch, contraction width, planner FMAs and bytes,
milliseconds (warm plan; plan build and first-call allocation excluded and reported separately), result.
The second half of BASELINE.json's metric ("time-to-exact E0+count"); the first half is bench.py.
No oracle here: correctness of the same instances is checked by tests/ (goldens written by the oracle).
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

from . import binding as bb
from . import instances as I

MASK64 = (1 << 64) - 1


def _sync():
    import torch
    torch.cuda.synchronize()


def _timed(fn, repeat):
    t0 = time.perf_counter(); out = fn(); _sync(); first = (time.perf_counter() - t0) * 1e3
    ts = []
    for _ in range(repeat):
        t0 = time.perf_counter(); out = fn(); _sync(); ts.append((time.perf_counter() - t0) * 1e3)
    return out, first, float(np.median(ts)), float(np.min(ts))


def _leaf_sum(kind, e, c):
    """Eq. 3's outer (+) over the leaf results, by the library (bbtn_oplus_combine)."""
    return bb.oplus_combine(kind, e, c)[:2]


def solve_unbranched(name, inst, tree=None, repeat=5, cap=1 << 28):
    h = bb.Handle(inst, tree=tree, max_elements_per_leaf=cap)
    info = h.plan_query(None, 1)
    (e, c), first, med, mn = _timed(lambda: h.contract_batch(), repeat)
    h.close()
    return {"instance": name, "mode": "unbranched", "n_vertices": inst.n_vertices, "n_edges": inst.n_edges,
            "width": info["max_rank"], "kernel_launches": info["n_kernel_launches"], "fma": info["fma_variant"] + info["fma_invariant"],
            "first_call_ms": first, "ms_median": med, "ms_min": mn, "energy": int(e[0]), "count_mod_2_64": int(c[0])}


def solve_branched(name, inst, fixed, tree, repeat=5, cap=1 << 26):
    assign = I.all_assignments(len(fixed))
    B = len(assign)
    h = bb.Handle(inst, tree=tree, max_elements_per_leaf=cap)
    info = h.plan_query(fixed, B)
    (e, c), first, med, mn = _timed(lambda: h.contract_batch(fixed, assign), repeat)
    h.close()
    best, cnt = _leaf_sum(inst.kind, e, c)
    fma = info["fma_variant"] * B + info["fma_invariant"]
    return {"instance": name, "mode": f"all 2^{len(fixed)} leaves of one fixed set, one bbtn_contract_batch call (host pointers)",
            "n_vertices": inst.n_vertices, "n_edges": inst.n_edges, "n_fixed": len(fixed), "leaves": B, "width": info["max_rank"],
            "nodes": info["n_nodes"], "variant_nodes": info["n_variant_nodes"], "fma": fma, "bytes": info["bytes_per_call"],
            "workspace_bytes": info["workspace_bytes"], "first_call_ms": first, "ms_median": med, "ms_min": mn,
            "gfma_per_s": fma / med / 1e6, "algorithmic_gb_per_s": info["bytes_per_call"] / med / 1e6,
            "energy": best, "count_mod_2_64": cnt}


def solve_king_bb(L, seed=1, block=4, chunk=4, max_batch=1024):
    k = I.kings_subgraph(L, L, 0.8, seed)
    ids = -np.ones((L, L), int)
    ids[k.meta["keep"]] = np.arange(k.n_vertices)
    offs, verts = [0], []
    for r0 in range(0, L, block):
        for c0 in range(0, L, block):
            verts += [int(ids[r][c]) for r in range(r0, min(r0 + block, L)) for c in range(c0, min(c0 + block, L)) if ids[r][c] >= 0]
            offs.append(len(verts))
    branch = np.array([ids[L // 2][c] for c in range(L) if ids[L // 2][c] >= 0], np.int32)
    h = bb.Handle(k, max_elements_per_leaf=1 << 26)
    t0 = time.perf_counter()
    out = h.solve_bb(branch, chunk, offs, verts, max_batch=max_batch, use_pruning=True)
    dt = time.perf_counter() - t0
    h.close()
    return {"instance": f"king {L}x{L} p0.8 seed {seed}", "mode": f"host B&B on the middle row ({len(branch)} vertices), {block}x{block} regions, K5 pruning",
            "n_vertices": k.n_vertices, "n_edges": k.n_edges, "seconds": dt, "energy": out["energy"], "count_mod_2_64": out["count"],
            "nodes_generated": out["generated"], "nodes_pruned": out["pruned"], "leaves_contracted": out["contracted"],
            "contract_calls": out["calls"]}


def solve_king_bbtn(L, seed=1, log2_target=31, crt=True):
    """BBTN proper (bbtn_solve_branching): rho-driven non-uniform branching, T_target = 2^log2_target elements."""
    k = I.kings_subgraph(L, L, 0.8, seed)
    h = bb.Handle(k, flags=bb.BBTN_COUNT_CRT if crt else 0)
    t0 = time.perf_counter()
    out = h.solve_branching(log2_target)
    dt = time.perf_counter() - t0
    h.close()
    cnt = bb.crt_combine(out["count"], *out["count_mod"]) if crt else out["count"]
    rings = 2 if crt else 1         # mod 2^64, then both primes packed in one 64-bit count
    return {"instance": f"king {L}x{L} p0.8 seed {seed}", "mode": f"BBTN branching on rho (Eq. 4), T_target = 2^{log2_target}"
            + (", counts mod 2^64 and mod (p1, p2), CRT-combined" if crt else ""),
            "n_vertices": k.n_vertices, "n_edges": k.n_edges, "seconds": dt, "energy": out["energy"],
            "count_mod_2_64": out["count"], "count": str(cnt), "rho_root": out["rho_root"], "branch_nodes": out["branch_nodes"],
            "leaves": out["leaves"], "max_fixed": out["max_fixed"], "fma": out["fma"] * rings, "bytes": out["bytes"] * rings,
            "algorithmic_gb_per_s": out["bytes"] * rings / dt / 1e9}


def solve_king_local(L, seed=1, log2_target=32, crt=True, block=4, hint=None, search=False):
    """BBTN on sub-networks (bbtn_solve_local): local fixed sets per overflowing stretch of the tree, K5 region bounds
    against the caller's incumbent (if any) on every branch."""
    k = I.kings_subgraph(L, L, 0.8, seed)
    ids = -np.ones((L, L), int)
    ids[k.meta["keep"]] = np.arange(k.n_vertices)
    offs, verts = [0], []
    for r0 in range(0, L, block):
        for c0 in range(0, L, block):
            verts += [int(ids[r][c]) for r in range(r0, min(r0 + block, L)) for c in range(c0, min(c0 + block, L)) if ids[r][c] >= 0]
            offs.append(len(verts))
    crt = crt and not search
    h = bb.Handle(k, flags=bb.BBTN_SEARCH_ONLY if search else (bb.BBTN_COUNT_CRT if crt else 0))
    h.add_sweep_order(I.column_major_order(k))          # the library also tries sweeps along the columns
    t0 = time.perf_counter()
    plan = h.local_plan_query(log2_target)
    t_plan = time.perf_counter() - t0
    t0 = time.perf_counter()
    out = h.solve_local(log2_target, region_offsets=offs, region_vertices=verts,
                        incumbent_hint=bb.BBTN_NEG_INF if hint is None else hint)
    dt = time.perf_counter() - t0
    h.close()
    cnt = bb.crt_combine(out["count"], *out["count_mod"]) if crt else out["count"]
    rings = 2 if crt else 1                             # mod 2^64, then both primes packed in one 64-bit count: 12 B/element each
    return {"instance": f"king {L}x{L} p0.8 seed {seed}", "mode": f"BBTN on sub-networks (bbtn_solve_local), T_target = 2^{log2_target}"
            + (", counts mod 2^64, then (p1, p2) packed (2 passes) CRT-combined" if crt else "")
            + (", search mode (energy plane only, 4 B per element; the count reads 0)" if search else ""),
            "n_vertices": k.n_vertices, "n_edges": k.n_edges, "seconds": dt, "plan_only_seconds": t_plan, "energy": out["energy"],
            "count_mod_2_64": out["count"], "count": str(cnt), **{key: out[key] for key in bb.Handle._LOCAL_STATS},
            "fma": out["fma"] * rings, "bytes": out["bytes"] * rings,
            "bytes_contracted": out["bytes_contracted"] * rings,
            "algorithmic_gb_per_s": out["bytes_contracted"] * rings / dt / 1e9}


def solve_e1(L, seed=1, log2_target=32):
    """The paper's spin-glass setting (+-J, field 0.5 -> 2J, h = 1, half units) unbranched: one leaf of width L+1."""
    inst = I.ising_lattice_2d_half_field(L, L, seed)
    h = bb.Handle(inst)
    t0 = time.perf_counter()
    out = h.solve_branching(log2_target)
    dt = time.perf_counter() - t0
    h.close()
    return {"instance": f"paper-E1 ising {L}x{L} seed {seed} h=0.5 (2J, h=1)", "mode": f"bbtn_solve_branching, T_target = 2^{log2_target}",
            "n_vertices": inst.n_vertices, "n_edges": inst.n_edges, "seconds": dt, "energy_half_units": out["energy"],
            "energy": out["energy"] / 2, "count_mod_2_64": out["count"], "leaves": out["leaves"], "rho_root": out["rho_root"],
            "fma": out["fma"], "bytes": out["bytes"], "algorithmic_gb_per_s": out["bytes"] / dt / 1e9}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", nargs="*", default=["1", "2", "3", "4b", "5"])
    ap.add_argument("--king-sizes", nargs="*", type=int, default=[16, 20, 24])
    ap.add_argument("--bbtn", nargs="*", default=[], help="L:seed:log2_target[:crt] runs of bbtn_solve_branching, e.g. 32:1:31:1")
    ap.add_argument("--local", nargs="*", default=[], help="L:seed:log2_target[:mode] runs of bbtn_solve_local, mode 0 = mod 2^64, 1 = CRT, 2 = search; e.g. 40:1:32:1")
    ap.add_argument("--e1", nargs="*", type=int, default=[], help="lattice sizes L for the paper's +-J, h = 0.5 setting, unbranched")
    ap.add_argument("--repeat", type=int, default=5)
    a = ap.parse_args()
    bb.load()
    emit = lambda d: print(json.dumps(d), flush=True)
    if "1" in a.configs:
        for seed in (1, 2, 3):
            emit(solve_unbranched(f"config1 ising 6x6 seed {seed}", I.ising_lattice_2d(6, 6, seed), repeat=a.repeat))
    if "2" in a.configs:
        for seed in (1, 2, 3):
            emit(solve_unbranched(f"config2 king 12x12 p0.8 seed {seed}", I.kings_subgraph(12, 12, 0.8, seed), repeat=a.repeat))
    if "3" in a.configs:
        inst = I.ising_lattice_2d(24, 24, 1)
        for f in (8, 10, 12):
            fixed = I.slit_fixed_set_2d(24, 24, f)
            tree = I.elimination_tree(inst.input_index_sets(fixed), I.slit_angular_order_2d(24, 24, f))
            emit(solve_branched("config3 ising 24x24 seed 1", inst, fixed, tree, repeat=a.repeat))
    if "4b" in a.configs:
        inst = I.ising_lattice_3d(5, 5, 5, 1)
        for f in (6, 8, 10):
            fixed = I.layer_fixed_set_3d(5, 5, 5, f)
            tree = I.elimination_tree(inst.input_index_sets(fixed), I.min_degree_order(inst, fixed))
            emit(solve_branched("config4b ising 5x5x5 seed 1", inst, fixed, tree, repeat=a.repeat))
    if "5" in a.configs:
        for L in a.king_sizes:
            emit(solve_king_bb(L))
    for L in a.e1:
        emit(solve_e1(L))
    for spec in a.local:
        f = [int(x) for x in spec.split(":")]
        emit(solve_king_local(f[0], f[1], f[2], crt=len(f) > 3 and f[3] == 1, search=len(f) > 3 and f[3] == 2))
    for spec in a.bbtn:
        f = [int(x) for x in spec.split(":")]
        emit(solve_king_bbtn(f[0], f[1], f[2], crt=bool(f[3]) if len(f) > 3 else False))


if __name__ == "__main__":
    main()
