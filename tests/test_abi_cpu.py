"""CPU-side checks of the boundary: the C-ABI library builds/loads, exports every symbol that
include/bbtn.h declares, validates its arguments, plans on the host, and refuses to compute
without a device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2602_05470_b200 import binding as bb
from paper_2602_05470_b200 import build as bbuild
from paper_2602_05470_b200 import instances as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    bbuild.build()
    return bb.load()


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "bbtn.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bbtn_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(bb.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.bbtn_version()


def test_build_validates_arguments(lib):
    inst = I.ising_lattice_2d(3, 3, 1)
    bb.Handle(inst).close()
    bad = I.ising_lattice_2d(3, 3, 1); bad.edge_v = bad.edge_v.copy(); bad.edge_v[0] = 99
    with pytest.raises(bb.BbtnError) as e:
        bb.Handle(bad)
    assert e.value.status == bb.BBTN_EINVAL
    dup = I.ising_lattice_2d(3, 3, 1); dup.edge_u = np.append(dup.edge_u, dup.edge_v[0]).astype(np.int32)
    dup.edge_v = np.append(dup.edge_v, dup.edge_u[0]).astype(np.int32); dup.edge_w = np.append(dup.edge_w, 1).astype(np.int32)
    with pytest.raises(bb.BbtnError) as e:
        bb.Handle(dup)
    assert e.value.status == bb.BBTN_EINVAL
    big = I.ising_lattice_2d(3, 3, 1); big.edge_w = (big.edge_w.astype(np.int64) * (1 << 27)).astype(np.int32)
    with pytest.raises(bb.BbtnError) as e:
        bb.Handle(big)
    assert e.value.status == bb.BBTN_ERANGE
    with pytest.raises(bb.BbtnError) as e:      # wrong number of tree steps
        bb.Handle(inst, tree=(np.zeros(3, np.int32), np.ones(3, np.int32)))
    assert e.value.status == bb.BBTN_EINVAL
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(9))
    tl2 = tl.copy(); tl2[5] = tl2[4]              # reuses a consumed tensor
    with pytest.raises(bb.BbtnError) as e:
        bb.Handle(inst, tree=(tl2, tr))
    assert e.value.status == bb.BBTN_EINVAL


def test_planner_widths_and_counts_on_host(lib):
    # row-major sweep of an LxL lattice has width L+1 (frontier L plus the new site's bond index)
    for L in (4, 6, 8):
        inst = I.ising_lattice_2d(L, L, 1)
        tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(L * L))
        h = bb.Handle(inst, tree=(tl, tr))
        info = h.plan_query()
        assert L <= info["max_rank"] <= L + 2
        assert info["n_variant_nodes"] == 0 and info["fma_variant"] == 0
        assert info["n_nodes"] == inst.n_edges + inst.n_vertices - 1
        assert info["rho"] == 0
        # fixing the middle column splits the lattice: width drops, nodes next to F become leaf-variant
        fixed = np.array([r * L + L // 2 for r in range(L)], np.int32)
        tl2, tr2 = I.elimination_tree(inst.input_index_sets(fixed), I.natural_order(L * L, exclude=fixed))
        h2 = bb.Handle(inst, tree=(tl2, tr2))
        info2 = h2.plan_query(fixed, B=16)
        assert info2["max_rank"] <= info["max_rank"]
        assert info2["n_variant_nodes"] > 0 and info2["fma_variant"] > 0
        # library-derived tree (tree = NULL) must also plan
        h3 = bb.Handle(inst)
        assert h3.plan_query(fixed, B=4)["max_rank"] >= 1


def test_rho_eq4_reported_when_cap_exceeded(lib):
    inst = I.ising_lattice_2d(8, 8, 1)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(64))
    h = bb.Handle(inst, tree=(tl, tr), max_elements_per_leaf=1 << 6)
    info = h.plan_query()
    assert info["max_rank"] > 6 and info["rho"] > 0        # Eq. 4: cumulative overflow over T_target


def test_slit_order_gives_narrow_leaves(lib):
    # config 3 recipe: f contiguous spins of the middle column + angular order -> width ~ max(L/2, L-f)+1
    L = 24
    inst = I.ising_lattice_2d(L, L, 1)
    for f, wmax in ((8, 19), (10, 17), (12, 15)):
        fixed = I.slit_fixed_set_2d(L, L, f)
        order = I.slit_angular_order_2d(L, L, f)
        assert len(order) == L * L - f
        tl, tr = I.elimination_tree(inst.input_index_sets(fixed), order)
        h = bb.Handle(inst, tree=(tl, tr), max_elements_per_leaf=1 << 26)
        info = h.plan_query(fixed, B=1 << f)
        assert info["max_rank"] <= wmax, (f, info)
        assert info["rho"] == 0


@pytest.mark.skipif(_has_gpu(), reason="checks the no-device behaviour")
def test_no_cpu_fallback(lib):
    inst = I.ising_lattice_2d(3, 3, 1)
    h = bb.Handle(inst)
    with pytest.raises(bb.BbtnError) as e:
        h.contract_batch()
    assert e.value.status == bb.BBTN_ECUDA
    with pytest.raises(bb.BbtnError) as e:
        h.region_bound([0], [])
    assert e.value.status == bb.BBTN_ECUDA
    with pytest.raises(bb.BbtnError) as e:
        bb.int32_microbench(0, 10)
    assert e.value.status == bb.BBTN_ECUDA
    # the no-allocation K5 entry point: its size limit is checked before anything touches a device, and without a
    # device it fails like every other compute call
    offs, verts = np.array([0, 4, 9], np.int32), np.arange(9, dtype=np.int32)
    dummy = np.zeros(8, np.int32)
    with pytest.raises(bb.BbtnError) as e:
        h.region_bound_static(offs, verts, None, None, dummy, B=(1 << 19) + 1)
    assert e.value.status == bb.BBTN_ESHAPE and "static scratch" in str(e.value)
    with pytest.raises(bb.BbtnError) as e:
        h.region_bound_static(offs, verts, None, None, dummy, B=4)
    assert e.value.status == bb.BBTN_ECUDA
    with pytest.raises(bb.BbtnError) as e:
        h.region_bound_static(offs, verts, None, None, None, B=-1)
    assert e.value.status == bb.BBTN_EINVAL


def test_crt_combine_host():
    for x in (0, 1, 2 ** 64 - 1, 2 ** 64 + 12345, 3 ** 70, 2 ** 125 + 7):
        got = bb.crt_combine(x % 2 ** 64, x % bb.BBTN_P1, x % bb.BBTN_P2)
        assert got == x


# ---- branching driver (host side of BBTN proper): rho-driven non-uniform leaves ----
@pytest.mark.parametrize("name,make,t", [
    ("king8", lambda: I.kings_subgraph(8, 8, 0.8, 1), 5),
    ("king10", lambda: I.kings_subgraph(10, 10, 0.8, 2), 6),
    ("king7w", lambda: I.kings_subgraph(7, 6, 0.9, 3), 6),
    ("ising5", lambda: I.ising_lattice_2d(5, 5, 3), 3),
    ("cube3", lambda: I.ising_lattice_3d(3, 3, 3, 2), 5),
])
def test_branching_leaves_are_complete_and_orthogonal(lib, oracle, name, make, t):
    """the decomposition must be complete and orthogonal, so the (+) over the leaves -- each
    evaluated by the ORACLE here -- reproduces the unbranched result; every leaf obeys rho = 0 (Eq. 4)."""
    inst = make()
    h = bb.Handle(inst)
    leaves, st = h.branching_leaves(t)
    assert st["rho_root"] > 0 and st["leaves"] == len(leaves) == st["branch_nodes"] + 1
    res = []
    for f, x in leaves:
        assert len(set(f.tolist())) == len(f)
        res.append(oracle.frontier_dp(inst, fixed=f, assign=x))
    if inst.kind == "mis":                                     # MIS rules fix different subsets in different branches
        assert len({tuple(sorted(f.tolist())) for f, _ in leaves}) > 1
    tot = (oracle.oplus_max if inst.kind == "mis" else oracle.oplus_min)(res)
    assert tuple(tot) == tuple(oracle.frontier_dp(inst))
    # orthogonality stated directly: any two leaves disagree on a vertex both fix
    for i in range(len(leaves)):
        for j in range(i + 1, len(leaves)):
            a = dict(zip(leaves[i][0].tolist(), leaves[i][1].tolist()))
            assert any(v in a and a[v] != x for v, x in zip(leaves[j][0].tolist(), leaves[j][1].tolist()))
    h.close()


def test_branching_target_above_width_is_one_leaf_and_guards(lib):
    inst = I.kings_subgraph(8, 8, 0.8, 1)
    h = bb.Handle(inst)
    leaves, st = h.branching_leaves(20)
    assert st["leaves"] == 1 and st["rho_root"] == 0 and len(leaves[0][0]) == 0
    with pytest.raises(bb.BbtnError):
        h.branching_leaves(3, max_leaves=2)            # needs more leaves than allowed -> ESHAPE
    with pytest.raises(bb.BbtnError):
        h.branching_leaves(0)                          # log2_target out of range
    h.close()


def test_crt_combine_matches_big_integers(lib):
    # bbtn_crt_combine is host arithmetic behind the ABI (reading A9): compare with Python's big integers
    P1, P2 = bb.BBTN_P1, bb.BBTN_P2
    M = (1 << 64) * P1 * P2
    vals = [0, 1, (1 << 64) - 1, 1 << 64, 6 ** 30, 2 ** 100, 4 ** 40 * 3, M - 1, 113847283001211021991799704166400]
    x = 0x9E3779B97F4A7C15
    for _ in range(200):
        x = (x * 6364136223846793005 + 1442695040888963407) % (1 << 128)
        vals.append(x % M)
    for v in vals:
        assert bb.crt_combine(v % (1 << 64), v % P1, v % P2) == v
    with pytest.raises(bb.BbtnError) as e:
        bb.crt_combine(0, P1, 0)                 # residue not below its prime
    assert e.value.status == bb.BBTN_EINVAL


def test_raw_gemm_argument_checks_need_no_device(lib):
    # count_bits outside 1..64 and launches beyond 2^31-1 thread blocks are refused before any CUDA call
    z = C.c_void_p(16)
    rc = lib.bbtn_tropical_gemm_batched(1, 64, 64, 64, z, z, z, z, z, z, 0, 0, 4096, 0, 32, None)
    assert rc == bb.BBTN_EINVAL
    rc = lib.bbtn_tropical_gemm_batched(1 << 40, 64, 64, 64, z, z, z, z, z, z, 0, 0, 4096, 64, 32, None)
    assert rc == bb.BBTN_ESHAPE
    rc = lib.bbtn_tropical_gemm_batched(1, 64, 64, 64, z, z, z, z, z, z, 0, 0, 4096, 64, 0, None)
    assert rc == bb.BBTN_EINVAL
    rc = lib.bbtn_tropical_gemm_batched(1 << 40, 64, 64, 64, z, z, z, z, z, z, 0, 0, 4096, 64, 32, None)
    assert rc == bb.BBTN_ESHAPE
    assert bb.set_debug_checks(False) in (False, True)


def test_block_tree_plans_use_tiled_gemm_and_trace(lib):
    # a divide-and-conquer tree makes the planner pick permute + tiled GEMM and the long-reduction kernel in
    # AUTOMATIC mode (the frontier sweeps of the lattice configs never do)
    inst = I.ising_lattice_2d(12, 12, 3)
    tree = I.grouped_elimination_tree(inst.input_index_sets(), I.lattice_block_parts(12, 12, [6], [6]))
    info = bb.Handle(inst, tree=tree).plan_query()
    assert info["n_gemm_tiled"] == 2 and info["n_permute"] >= 2 and info["n_trace"] == 1
    assert info["n_nodes"] == inst.n_edges + inst.n_vertices - 1


def test_small_subtrees_become_a_prologue_and_mid_sized_operands_are_relaid_on_host(lib):
    # host logic of the launch plan (no device): the small subtrees of the 5x5x5 cube's leaves collapse into one or two
    # shared-memory launches (api.cu prepare_hybrid) and the planner re-lays the mid-sized gathered operands of its large
    # nodes (K2 steps in a tree that has no tiled GEMM); BBTN_NO_FUSED keeps one launch per node.  The totals the planner
    # reports for the tree itself (nodes, FMAs) do not depend on how it is launched.
    inst = I.ising_lattice_3d(5, 5, 5, 1)
    fixed = I.layer_fixed_set_3d(5, 5, 5, 8)
    tree = I.elimination_tree(inst.input_index_sets(fixed), I.min_degree_order(inst, fixed))
    hyb = bb.Handle(inst, tree=tree).plan_query(fixed, 256)
    per_node = bb.Handle(inst, tree=tree, flags=bb.BBTN_NO_FUSED).plan_query(fixed, 256)
    assert hyb["n_nodes"] == per_node["n_nodes"] == 407 and hyb["fma_variant"] == per_node["fma_variant"]
    assert hyb["n_gemm_tiled"] == 0 and hyb["n_permute"] > 0
    assert per_node["n_kernel_launches"] == per_node["n_nodes"] + per_node["n_permute"] + 4
    assert hyb["n_kernel_launches"] < 80
    # the prologue's outputs get fresh storage behind the planned arenas: a little more workspace, never less
    assert per_node["workspace_bytes"] <= hyb["workspace_bytes"] <= 1.02 * per_node["workspace_bytes"]
    # a small network (every tensor of a leaf fits shared memory) is left to the one-launch form
    small = bb.Handle(I.kings_subgraph(12, 12, 0.8, 1)).plan_query()
    assert small["n_kernel_launches"] > small["n_nodes"] and small["n_permute"] == 0


def test_local_plan_query_and_sweep_order_hints_on_host(lib):
    # bbtn_local_plan_query / bbtn_add_sweep_order need no device: a King's subgraph whose sweep is wider than the threshold
    # gets sliced stretches with small local fixed sets; a hinted order is validated and can only make the plan cheaper
    k = I.kings_subgraph(14, 14, 0.8, 5)
    h = bb.Handle(k)
    wide = h.local_plan_query(30)
    assert wide["sliced_stretches"] == 0 and wide["branches_planned"] == 1 and wide["max_fixed"] == 0
    q = h.local_plan_query(wide["max_rank"] - 2)
    assert q["sliced_stretches"] >= 1 and 1 <= q["max_fixed"] <= 24 and q["max_rank"] <= wide["max_rank"] - 2
    assert q["branches_planned"] > q["stretches"] - q["sliced_stretches"] and q["bytes"] > 0
    with pytest.raises(bb.BbtnError) as e:
        h.add_sweep_order(np.zeros(k.n_vertices, np.int32))
    assert e.value.status == bb.BBTN_EINVAL
    h.add_sweep_order(I.column_major_order(k))
    q2 = h.local_plan_query(wide["max_rank"] - 2)
    assert q2["bytes"] <= q["bytes"] and q2["max_rank"] <= wide["max_rank"] - 2
    with pytest.raises(bb.BbtnError):
        h.local_plan_query(0)
