"""Pins for the CPU oracle (oracle/): every function is checked against something
other than itself -- values worked by hand / fixed by the paper's definitions
(tests/golden/closed_forms.json), closed forms, invariants, brute force on tiny
inputs and library routines (numpy).  CPU only."""
import itertools
import json
import os

import numpy as np
import pytest

from paper_2602_05470_b200 import instances as I

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.json")))


def _inst(kind, n, edges, ew, vw):
    eu = np.array([e[0] for e in edges], np.int32)
    ev = np.array([e[1] for e in edges], np.int32)
    return I.Instance(kind, n, eu, ev, None if ew is None else np.array(ew, np.int32),
                      None if vw is None else np.array(vw, np.int32))


def _all3(oracle, inst, fixed=None, assign=None, order_seed=0):
    """(exhaustive, tree contraction, frontier DP) on one instance."""
    free_order = I.natural_order(inst.n_vertices, exclude=() if fixed is None else fixed)
    tl, tr = I.elimination_tree(inst.input_index_sets(() if fixed is None else fixed), free_order)
    a = oracle.exhaustive(inst, fixed, assign)
    b = oracle.contract_tree(inst, tl, tr, fixed, assign)
    c = oracle.frontier_dp(inst, None, fixed, assign)
    return a, b, c


# ---- the PRNG the generators are built on -------------------------------------
def test_splitmix64_reference_vector():
    # published SplitMix64 test vector for seed 0
    got = [int(x) for x in I.splitmix64(0, 4)]
    assert got == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F, 0xF88BB8A8724C81EC]
    assert int(I.splitmix64(0, 10)[7]) == int(I.splitmix64(0, 8)[7])     # counter-based


# ---- hand-worked values ---------------------------------------------------------
@pytest.mark.parametrize("case", GOLD["ising"], ids=lambda c: c["name"])
def test_ising_hand_values(oracle, case):
    inst = _inst("ising", case["n"], case["edges"], case["J"], case["h"])
    for got in _all3(oracle, inst):
        assert got == (case["E0"], case["count"])


@pytest.mark.parametrize("case", GOLD["mis"], ids=lambda c: c["name"])
def test_mis_hand_values(oracle, case):
    inst = _inst("mis", case["n"], case["edges"], None, case["w"])
    for got in _all3(oracle, inst):
        assert got == (case["size"], case["count"])


# ---- closed forms -----------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 3, 4])
def test_ferromagnet_closed_form_all_oracles(oracle, L):
    # north_star: all-+J LxL open lattice has E0 = -2L(L-1), degeneracy 2
    inst = I.ising_lattice_2d(L, L, seed=1, ferro=True)
    for got in _all3(oracle, inst):
        assert got == (-2 * L * (L - 1), 2)


@pytest.mark.parametrize("L", [6, 9, 12])
def test_ferromagnet_closed_form_large(oracle, L):
    inst = I.ising_lattice_2d(L, L, seed=1, ferro=True)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(L * L))
    assert oracle.contract_tree(inst, tl, tr) == (-2 * L * (L - 1), 2)
    assert oracle.frontier_dp(inst) == (-2 * L * (L - 1), 2)
    # all -J on a bipartite lattice is gauge-equivalent
    inst.edge_w = -inst.edge_w
    assert oracle.contract_tree(inst, tl, tr) == (-2 * L * (L - 1), 2)


@pytest.mark.parametrize("n,seed", [(5, 1), (12, 2), (40, 3)])
def test_pm_j_chain_closed_form(oracle, n, seed):
    # any tree with +-J bonds is unfrustrated: E0 = -|E|, count 2
    inst = I.ising_lattice_2d(1, n, seed)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(n))
    assert oracle.contract_tree(inst, tl, tr) == (-(n - 1), 2)
    assert oracle.frontier_dp(inst) == (-(n - 1), 2)


@pytest.mark.parametrize("case", GOLD["kings_full"], ids=lambda c: f"L{c['L']}")
def test_full_kings_grid(oracle, case):
    L = case["L"]
    k = I.kings_subgraph(L, L, 1.0, seed=1)
    assert k.n_vertices == L * L
    tl, tr = I.elimination_tree(k.input_index_sets(), I.natural_order(L * L))
    assert oracle.contract_tree(k, tl, tr) == (case["size"], case["count"])
    assert oracle.frontier_dp(k) == (case["size"], case["count"])
    if L <= 4:
        assert oracle.exhaustive(k) == (case["size"], case["count"])


@pytest.mark.parametrize("n", [1, 2, 5, 6, 9, 10])
def test_mis_path_cycle_complete_edgeless(oracle, n):
    path = _inst("mis", n, [(i, i + 1) for i in range(n - 1)], None, None)
    want = ((n + 1) // 2, 1 if n % 2 else n // 2 + 1)
    for got in _all3(oracle, path):
        assert got == want
    if n >= 3:
        cyc = _inst("mis", n, [(i, (i + 1) % n) for i in range(n)], None, None)
        want = (n // 2, 2) if n % 2 == 0 else ((n - 1) // 2, n)
        for got in _all3(oracle, cyc):
            assert got == want
    comp = _inst("mis", n, list(itertools.combinations(range(n), 2)), None, None)
    for got in _all3(oracle, comp):
        assert got == (1, n) if n > 1 else got == (1, 1)
    empty = _inst("mis", n, [], None, None)
    for got in _all3(oracle, empty):
        assert got == (n, 1)


def test_counts_beyond_2_64(oracle):
    # 100 isolated field-free spins: every configuration is a ground state: (0, 2^100)  (reading A7)
    inst = _inst("ising", 100, [], [], None)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(100))
    assert oracle.contract_tree(inst, tl, tr) == (0, 1 << 100)
    assert oracle.frontier_dp(inst) == (0, 1 << 100)
    # 40 disjoint copies of K4: (40, 4^40) -- exercises the 256-bit product
    edges = []
    for k in range(40):
        edges += [(4 * k + a, 4 * k + b) for a, b in itertools.combinations(range(4), 2)]
    inst = _inst("mis", 160, edges, None, None)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(160))
    assert oracle.contract_tree(inst, tl, tr) == (40, 4 ** 40)
    assert oracle.frontier_dp(inst) == (40, 4 ** 40)
    # 30 disjoint triangles with J=-1: energy -30, count 6^30 > 2^64
    edges = []
    for k in range(30):
        edges += [(3 * k, 3 * k + 1), (3 * k + 1, 3 * k + 2), (3 * k, 3 * k + 2)]
    inst = _inst("ising", 90, edges, [-1] * 90, None)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(90))
    assert oracle.contract_tree(inst, tl, tr) == (-30, 6 ** 30)


# ---- brute force: oracle-2 and oracle-3 against the definition ----------------------
@pytest.mark.parametrize("seed", range(8))
def test_tree_and_dp_equal_exhaustive_ising(oracle, seed):
    shapes = [(3, 3), (3, 4), (4, 4), (2, 7), (4, 5), (3, 6), (2, 2), (4, 6)]
    r, c = shapes[seed]
    inst = I.ising_lattice_2d(r, c, seed, field_h=(seed % 3) - 1)
    n = r * c
    want = oracle.exhaustive(inst)
    for oseed in range(2):
        order = I.random_order(n, 100 + oseed)
        tl, tr = I.elimination_tree(inst.input_index_sets(), order)
        assert oracle.contract_tree(inst, tl, tr) == want
        assert oracle.frontier_dp(inst, order) == want
    tl, tr = I.sequential_tree(inst.n_edges + n) if n <= 12 else I.elimination_tree(inst.input_index_sets(), I.natural_order(n))
    assert oracle.contract_tree(inst, tl, tr) == want


@pytest.mark.parametrize("seed", range(6))
def test_random_graphs_with_fields_and_weights(oracle, seed):
    gi = I.random_graph(11 + seed, 0.3, seed, "ising", field_h=True)
    gm = I.random_graph(12 + seed, 0.25, seed, "mis")
    for inst in (gi, gm):
        a, b, c = _all3(oracle, inst)
        assert a == b == c
        assert a[1] >= 1


@pytest.mark.parametrize("seed", range(5))
def test_cubes_and_kings(oracle, seed):
    cube = I.ising_lattice_3d(2, 3, 2 + seed % 2, seed)
    a, b, c = _all3(oracle, cube)
    assert a == b == c
    k = I.kings_subgraph(4, 5, [0.6, 0.8, 0.9, 1.0, 0.7][seed], seed, weights="unit" if seed % 2 else "rand")
    a, b, c = _all3(oracle, k)
    assert a == b == c


@pytest.mark.parametrize("seed", range(6))
def test_sliced_leaves_equal_exhaustive(oracle, seed):
    # Eq. 3: a leaf fixes s_{V_f} = x; minimise/count over the free variables only
    inst = I.ising_lattice_2d(4, 4, seed) if seed % 2 == 0 else I.kings_subgraph(4, 5, 0.8, seed)
    n = inst.n_vertices
    f = 1 + seed % 4
    fixed = I.random_order(n, 50 + seed)[:f]
    for x in I.random_assignments(4, f, seed):
        a, b, c = _all3(oracle, inst, fixed, x)
        assert a == b == c


def test_infeasible_mis_leaf_is_zero_element(oracle):
    # hard constraint = tuple (inf, 0): two adjacent vertices fixed to 1
    k = I.kings_subgraph(3, 3, 1.0, 1)
    fixed = np.array([0, 1], np.int32)
    for got in _all3(oracle, k, fixed, [1, 1]):
        assert got == (None, 0)
    for got in _all3(oracle, k, fixed, [1, 0]):
        assert got[0] is not None and got[1] >= 1


# ---- invariants ---------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(4))
def test_ising_invariants(oracle, seed):
    inst = I.ising_lattice_2d(5, 5, seed)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(25))
    e0, cnt = oracle.contract_tree(inst, tl, tr)
    assert cnt >= 1 and cnt % 2 == 0                       # global flip symmetry, h = 0
    assert -inst.n_edges <= e0 <= 0
    assert (e0 - inst.n_edges) % 2 == 0                    # |J| = 1: H = |E| - 2*(satisfied bonds)... parity of |E|
    # gauge invariance: flip every bond at one vertex
    v = 7 + seed
    g = I.ising_lattice_2d(5, 5, seed)
    touch = (g.edge_u == v) | (g.edge_v == v)
    g.edge_w = np.where(touch, -g.edge_w, g.edge_w).astype(np.int32)
    assert oracle.contract_tree(g, tl, tr) == (e0, cnt)
    assert oracle.frontier_dp(g) == (e0, cnt)


@pytest.mark.parametrize("seed", range(4))
def test_eq3_leaf_sum_reproduces_unbranched(oracle, seed):
    # Eq. 3: (+) over all 2^f assignments of the sliced contractions == unsliced
    if seed % 2 == 0:
        inst, red = I.ising_lattice_2d(4, 5, seed), oracle.oplus_min
    else:
        inst, red = I.kings_subgraph(5, 5, 0.8, seed), oracle.oplus_max
    n = inst.n_vertices
    tl0, tr0 = I.elimination_tree(inst.input_index_sets(), I.natural_order(n))
    whole = oracle.contract_tree(inst, tl0, tr0)
    f = 3
    fixed = I.random_order(n, 9 + seed)[:f]
    tl, tr = I.elimination_tree(inst.input_index_sets(fixed), I.natural_order(n, exclude=fixed))
    leaves = [oracle.contract_tree(inst, tl, tr, fixed, x) for x in I.all_assignments(f)]
    assert red(leaves) == whole
    # a complete + orthogonal NON-uniform decomposition: {v0=0} u {v0=1,v1=0} u {v0=1,v1=1}
    parts = [(fixed[:1], [0]), (fixed[:2], [1, 0]), (fixed[:2], [1, 1])]
    leaves = [oracle.frontier_dp(inst, None, fx, x) for fx, x in parts]
    assert red(leaves) == whole


def test_tree_independence_same_tree_unsliced_on_sliced(oracle):
    # the SAME full-network tree must work when inputs are sliced (rank-0 inputs stay in the tree)
    inst = I.ising_lattice_2d(4, 4, 5)
    tl, tr = I.elimination_tree(inst.input_index_sets(), I.natural_order(16))
    fixed = np.array([5, 6, 9], np.int32)
    for x in I.all_assignments(3):
        assert oracle.contract_tree(inst, tl, tr, fixed, x) == oracle.exhaustive(inst, fixed, x)


# ---- raw GEMM ---------------------------------------------------------------------------
def _el(x):
    return (0, 1, 0) if x[0] == "z" else (x[0], 0, x[1])


def test_gemm_worked_example(oracle):
    g = GOLD["gemm_2x2"]
    A = np.array([[_el(x) for x in row] for row in g["A"]])
    B = np.array([[_el(x) for x in row] for row in g["B"]])
    Ce, Cz, Cc = oracle.gemm(A[None, :, :, 0], A[None, :, :, 1], A[None, :, :, 2],
                             B[None, :, :, 0], B[None, :, :, 1], B[None, :, :, 2])
    want = np.array(g["C"])
    assert (Cz == 0).all()
    assert (Ce[0] == want[:, :, 0]).all() and (Cc[0] == want[:, :, 1].astype(np.uint64)).all()


def test_gemm_zero_energy_is_integer_matmul(oracle):
    # all energies equal => every k ties => counts are the ordinary matrix product mod 2^64 (numpy)
    Ae, Ac, Be, Bc = I.gemm_operands(2, 9, 7, 13, seed=3, wide_counts=True)
    z = np.zeros_like
    Ce, Cz, Cc = oracle.gemm(z(Ae), z(Ae), Ac, z(Be), z(Be), Bc)
    with np.errstate(over="ignore"):
        want = np.matmul(Ac, Bc)          # uint64 wraps mod 2^64
    assert (Cc == want).all() and (Ce == 0).all() and (Cz == 0).all()
    # full-width counts: compare with Python big integers
    _, _, _, Cc4 = oracle.gemm(z(Ae), z(Ae), Ac, z(Be), z(Be), Bc, full_counts=True)
    big = sum(int(Ac[0, 1, k]) * int(Bc[0, k, 2]) for k in range(13))
    got = sum(int(Cc4[0, 1, 2, l]) << (64 * l) for l in range(4))
    assert got == big


def test_gemm_energies_are_textbook_maxplus(oracle):
    Ae, Ac, Be, Bc = I.gemm_operands(3, 17, 11, 23, seed=4)
    Ce, Cz, Cc = oracle.gemm(Ae, np.zeros_like(Ae), Ac, Be, np.zeros_like(Be), Bc)
    want = (Ae[:, :, :, None].astype(np.int64) + Be[:, None, :, :]).max(axis=2)
    assert (Ce == want).all()
    # counts: sum over the argmax set of products (numpy restatement with masks)
    tie = (Ae[:, :, :, None].astype(np.int64) + Be[:, None, :, :]) == want[:, :, None, :]
    wantc = (tie * (Ac[:, :, :, None] * Bc[:, None, :, :])).sum(axis=2, dtype=np.uint64)
    assert (Cc == wantc).all()


def test_gemm_identity_and_associativity(oracle):
    n = 12
    Ae, Ac, Be, Bc = I.gemm_operands(1, n, n, n, seed=5, neg_inf_frac=0.2)
    Az = (Ac == 0).astype(np.uint8); Bz = (Bc == 0).astype(np.uint8)
    Ie = np.zeros((1, n, n), np.int64); Iz = 1 - np.eye(n, dtype=np.uint8)[None]; Ic = np.eye(n, dtype=np.uint64)[None]
    Ce, Cz, Cc = oracle.gemm(Ae, Az, Ac, Ie, Iz, Ic)
    assert (Cz == Az).all() and (Cc == Ac).all() and (np.where(Az == 1, 0, Ae) == Ce).all()
    De, Dz, Dc = oracle.gemm(Ae, Az, Ac, Be, Bz, Bc)
    Xe, Xc = I.gemm_operands(1, n, n, n, seed=7)[0:2]
    Xz = np.zeros_like(Xe, dtype=np.uint8)
    l = oracle.gemm(De, Dz, Dc, Xe, Xz, Xc)                      # (A B) X
    BXe, BXz, BXc = oracle.gemm(Be, Bz, Bc, Xe, Xz, Xc)
    r = oracle.gemm(Ae, Az, Ac, BXe, BXz, BXc)                   # A (B X)
    for a, b in zip(l, r):
        assert (a == b).all()


def test_gemm_zero_rows_give_zero_element(oracle):
    Ae, Ac, Be, Bc = I.gemm_operands(1, 4, 4, 4, seed=8)
    Az = np.zeros_like(Ae, dtype=np.uint8); Az[0, 2, :] = 1
    Ce, Cz, Cc = oracle.gemm(Ae, Az, Ac, Be, np.zeros_like(Be, dtype=np.uint8), Bc)
    assert (Cz[0, 2] == 1).all() and (Cc[0, 2] == 0).all() and Cz.sum() == 4


# ---- permute ------------------------------------------------------------------------------
@pytest.mark.parametrize("r,seed", [(1, 0), (4, 1), (9, 2), (12, 3)])
def test_permute_against_numpy_transpose(oracle, r, seed):
    perm = I.random_bit_permutation(r, seed)
    n = 1 << r
    src_e = (I.splitmix64(seed, 2 * n, 8) % np.uint64(1000)).astype(np.int32).reshape(2, n)
    src_c = I.splitmix64(seed, 2 * n, 9).reshape(2, n)
    dst_e, dst_c = oracle.permute(perm, src_e, src_c)
    # numpy: axis a of the reshaped array <-> bit (r-1-a); dst bit j takes src bit perm[j]
    axes = [0] + [1 + (r - 1 - int(perm[r - 1 - a])) for a in range(r)]
    want_e = src_e.reshape([2] + [2] * r).transpose(axes).reshape(2, n)
    want_c = src_c.reshape([2] + [2] * r).transpose(axes).reshape(2, n)
    assert (dst_e == want_e).all() and (dst_c == want_c).all()
    inv = np.argsort(perm).astype(np.int32)
    back_e, back_c = oracle.permute(inv, dst_e, dst_c)
    assert (back_e == src_e).all() and (back_c == src_c).all()


# ---- region bound (reading A15) and Eq. 4 ----------------------------------------------------
def _regions_grid(rows, cols, br, bc, ids=None):
    offs, verts = [0], []
    for r0 in range(0, rows, br):
        for c0 in range(0, cols, bc):
            for r in range(r0, min(r0 + br, rows)):
                for c in range(c0, min(c0 + bc, cols)):
                    v = r * cols + c if ids is None else ids[r][c]
                    if v >= 0:
                        verts.append(v)
            offs.append(len(verts))
    return np.array(offs, np.int32), np.array(verts, np.int32)


def test_region_bound_hand_example(oracle):
    # 4-cycle with one negative bond, h = 0.  No regions: every bond contributes |J| -> bound 4 (exact is 2).
    inst = _inst("ising", 4, [(0, 1), (1, 2), (2, 3), (3, 0)], [1, 1, 1, -1], None)
    assert oracle.region_bound(inst, [0], []) == 4
    # one region holding everything: bound is exact, -E0 = 2
    assert oracle.region_bound(inst, [0, 4], [0, 1, 2, 3]) == 2
    # regions {0,1},{2,3}: inside bonds (0,1),(2,3) satisfiable -> 1+1, crossing bonds uncovered -> 1+1
    assert oracle.region_bound(inst, [0, 2, 4], [0, 1, 2, 3]) == 4
    # fix spin 0 = +1, 3 = +1 (bond (3,0) J=-1 contributes -1); region {1,2}: bonds (0,1),(1,2),(2,3) all satisfiable: 3
    assert oracle.region_bound(inst, [0, 2], [1, 2], [0, 3], [1, 1]) == 2
    # MIS triangle, no regions: 3 (every vertex may be in); one region: exact 1; vertex 0 fixed in: 1 + 0 + 0
    tri = _inst("mis", 3, [(0, 1), (1, 2), (0, 2)], None, None)
    assert oracle.region_bound(tri, [0], []) == 3
    assert oracle.region_bound(tri, [0, 3], [0, 1, 2]) == 1
    assert oracle.region_bound(tri, [0], [], [0], [1]) == 1
    assert oracle.region_bound(tri, [0], [], [0, 1], [1, 1]) is None


@pytest.mark.parametrize("seed", range(6))
def test_region_bound_is_admissible_and_tight_when_covering(oracle, seed):
    if seed % 2 == 0:
        rows, cols = 4, 5
        inst = I.ising_lattice_2d(rows, cols, seed, field_h=seed % 3 - 1)
        ids = None
    else:
        rows, cols = 4, 5
        inst = I.kings_subgraph(rows, cols, 0.85, seed)
        ids = -np.ones((rows, cols), int); ids[inst.meta["keep"]] = np.arange(inst.n_vertices)
    n = inst.n_vertices
    fixed = I.random_order(n, 77 + seed)[:3]
    offs, verts = _regions_grid(rows, cols, 2, 2, ids)
    whole = (np.array([0, n], np.int32), np.arange(n, dtype=np.int32))
    for x in I.all_assignments(3):
        e, c = oracle.exhaustive(inst, fixed, x)
        b = oracle.region_bound(inst, offs, verts, fixed, x)
        bw = oracle.region_bound(inst, whole[0], whole[1], fixed, x)
        if e is None:
            assert b is None and bw is None
            continue
        exact = -e if inst.kind == "ising" else e
        assert b is not None and b >= exact       # admissible
        assert bw == exact                        # regions cover V\F, nothing uncovered -> tight


def test_rho_eq4(oracle):
    # Eq. 4: rho = sum_T max(0, log2|T| - log2 T_target)
    assert oracle.rho([10, 31, 33, 35, 2], 31) == 2 + 4
    assert oracle.rho([5, 6], 31) == 0


# ---- oracle-3, sparse MIS form (only independent frontier states stored) ------------------------
@pytest.mark.parametrize("L,p,seed", [(3, 1.0, 1), (4, 1.0, 1), (5, 0.8, 1), (4, 0.7, 2), (3, 0.5, 3)])
def test_sparse_mis_dp_equals_exhaustive(oracle, L, p, seed):
    inst = I.kings_subgraph(L, L + 1, p, seed)          # <= 24 vertices: the definition itself
    assert oracle.frontier_dp_mis_sparse(inst) == oracle.exhaustive(inst)


@pytest.mark.parametrize("case", GOLD["kings_full"], ids=lambda c: f"L{c['L']}")
def test_sparse_mis_dp_full_kings_closed_form(oracle, case):
    # north_star: a full odd-L King's grid has MIS size ((L+1)/2)^2 and count 1; 4x4 -> (4, 79)
    inst = I.kings_subgraph(case["L"], case["L"], 1.0, 0)
    assert oracle.frontier_dp_mis_sparse(inst) == (case["size"], case["count"])


@pytest.mark.parametrize("L", [9, 11, 13])
def test_sparse_mis_dp_odd_full_grid(oracle, L):
    inst = I.kings_subgraph(L, L, 1.0, 0)
    assert oracle.frontier_dp_mis_sparse(inst) == (((L + 1) // 2) ** 2, 1)


@pytest.mark.parametrize("seed", range(4))
def test_sparse_mis_dp_equals_dense_dp_orders_weights_and_slices(oracle, seed):
    inst = I.kings_subgraph(7 + seed, 9, 0.8, seed)
    inst.vertex_w = (1 + (I.splitmix64(seed, inst.n_vertices, 7) % 3)).astype(np.int32)   # MWIS weights 1..3
    order = np.arange(inst.n_vertices, dtype=np.int32)[::-1].copy() if seed % 2 else None     # a second sweep direction
    assert oracle.frontier_dp_mis_sparse(inst, order=order) == oracle.frontier_dp(inst)
    fixed = I.random_order(inst.n_vertices, 100 + seed)[:5]
    for x in I.all_assignments(5)[:: 7]:
        assert oracle.frontier_dp_mis_sparse(inst, fixed=fixed, assign=x) == oracle.frontier_dp(inst, fixed=fixed, assign=x)


def test_sparse_mis_dp_path_and_cycle(oracle):
    # P_n: size ceil(n/2), count 1 (n odd) or n/2+1 (n even);  C_n: (n/2, 2) n even, ((n-1)/2, n) n odd
    for n in (7, 10, 31, 40):
        path = _inst("mis", n, [(i, i + 1) for i in range(n - 1)], None, None)
        assert oracle.frontier_dp_mis_sparse(path) == ((n + 1) // 2, 1 if n % 2 else n // 2 + 1)
        cyc = _inst("mis", n, [(i, (i + 1) % n) for i in range(n)], None, None)
        assert oracle.frontier_dp_mis_sparse(cyc) == ((n // 2, 2) if n % 2 == 0 else ((n - 1) // 2, n))


def test_block_trees_equal_exhaustive(oracle):
    # divide-and-conquer trees (instances.grouped_elimination_tree: blocks contracted to boundary tensors, then
    # joined) give the definition's result too: == exhaustive on <= 24 vertices, with and without a sliced leaf
    for rows, cols, rc, cc in ((4, 6, [2], [3]), (5, 4, [2], [2]), (3, 8, [], [3, 5])):
        inst = I.ising_lattice_2d(rows, cols, rows + cols, field_h=1)
        tree = I.grouped_elimination_tree(inst.input_index_sets(), I.lattice_block_parts(rows, cols, rc, cc))
        assert len(tree[0]) == inst.n_edges + inst.n_vertices - 1
        assert oracle.contract_tree(inst, *tree) == oracle.exhaustive(inst)
        fixed = np.array([1, cols + 1], np.int32)
        parts = I.lattice_block_parts(rows, cols, rc, cc, exclude=fixed)
        t2 = I.grouped_elimination_tree(inst.input_index_sets(fixed), parts)
        for x in I.all_assignments(2):
            assert oracle.contract_tree(inst, t2[0], t2[1], fixed, x) == oracle.exhaustive(inst, fixed, x)
    k = I.kings_subgraph(4, 6, 1.0, 1, weights="rand")
    tree = I.grouped_elimination_tree(k.input_index_sets(), I.lattice_block_parts(4, 6, [2], [3]))
    assert oracle.contract_tree(k, *tree) == oracle.exhaustive(k)
