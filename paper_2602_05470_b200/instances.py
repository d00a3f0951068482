"""Seeded synthetic input generators.

This module is the ONLY code shared by the CPU oracle's callers and the CUDA
path's callers (tests, bench.py, smoke()).  It holds none of the method's
arithmetic: no tropical algebra, no contraction, no bounds.  It produces
graphs, couplings, fixed sets, assignments, contraction *orders/trees* (pure
structure) and raw GEMM operands, all from one specified counter-based PRNG
(SplitMix64) so that every input is reproducible bit for bit.

Shapes and value distributions follow the paper's workloads
("coupling constants J randomly chosen as +1 or -1";
PAPER.md:77,83 "random KSG with filling rate 0.8", unit weight) and the
canonical orders fixed in SURVEY.md section 8(d).  These synthetic instances
stand in for the paper's own instances, which are not available.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_STREAM = np.uint64(0x632BE59BD9B4E019)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, n: int, stream: int = 0) -> np.ndarray:
    """n outputs of the standard SplitMix64 generator.

    Output i (0-based) is mix(state0 + (i+1)*GOLDEN) with
    state0 = seed + stream*0x632BE59BD9B4E019 (mod 2^64), i.e. for stream 0 it
    is exactly the reference SplitMix64 sequence of `seed`
    (seed 0 -> 0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F, ...).
    Counter-based: output i does not depend on n.
    """
    with np.errstate(over="ignore"):
        s0 = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + np.uint64(stream) * _STREAM
        z = s0 + (np.arange(1, n + 1, dtype=np.uint64) * _GOLDEN)
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


@dataclass
class Instance:
    """A problem instance in the C-ABI's own terms (include/bbtn.h)."""
    kind: str                      # "ising" | "mis"
    n_vertices: int
    edge_u: np.ndarray             # int32 [n_edges]
    edge_v: np.ndarray             # int32 [n_edges]
    edge_w: np.ndarray | None      # int32 [n_edges] couplings J_ij (ising) / None (mis)
    vertex_w: np.ndarray | None    # int32 [n_vertices] fields h_i (ising) / weights w_i (mis) / None
    meta: dict = field(default_factory=dict)

    @property
    def n_edges(self) -> int:
        return int(self.edge_u.shape[0])

    def input_index_sets(self, fixed=()) -> list[list[int]]:
        """Index sets of the input tensors in ABI order (edges, then vertices),
        with the indices in `fixed` sliced away (Eq. 3)."""
        fx = set(int(v) for v in fixed)
        sets = [[int(x) for x in (u, v) if int(x) not in fx]
                for u, v in zip(self.edge_u, self.edge_v)]
        sets += [[i] if i not in fx else [] for i in range(self.n_vertices)]
        return sets


def _pm1(seed: int, n: int, stream: int) -> np.ndarray:
    bits = splitmix64(seed, n, stream) >> np.uint64(63)
    return (2 * bits.astype(np.int64) - 1).astype(np.int32)


def ising_lattice_2d(rows: int, cols: int, seed: int, field_h: int = 0,
                     ferro: bool = False) -> Instance:
    """Open-boundary rows x cols +-J lattice.  Vertex id = r*cols + c; bonds are
    enumerated per site row-major, right neighbour then down neighbour; J_e is
    +1 iff the top bit of SplitMix64 output e (stream 0) is 1."""
    eu, ev = [], []
    for r in range(rows):
        for c in range(cols):
            if c + 1 < cols:
                eu.append(r * cols + c); ev.append(r * cols + c + 1)
            if r + 1 < rows:
                eu.append(r * cols + c); ev.append((r + 1) * cols + c)
    m = len(eu)
    J = np.ones(m, np.int32) if ferro else _pm1(seed, m, 0)
    h = None if field_h == 0 else np.full(rows * cols, field_h, np.int32)
    return Instance("ising", rows * cols, np.array(eu, np.int32), np.array(ev, np.int32), J, h,
                    {"shape": (rows, cols), "seed": seed})


def ising_lattice_2d_half_field(rows: int, cols: int, seed: int) -> Instance:
    """The paper's spin-glass setting (J = +-1 at random, external field 0.5) in integers
    (reading A6): every coupling doubled, h = 1, energies come out in HALF units."""
    inst = ising_lattice_2d(rows, cols, seed, field_h=1)
    inst.edge_w = (2 * inst.edge_w).astype(np.int32)
    inst.meta["energy_unit"] = 0.5
    return inst


def ising_lattice_3d(lx: int, ly: int, lz: int, seed: int) -> Instance:
    """Open-boundary cubic +-J lattice, id = (z*ly + y)*lx + x, bonds +x, +y, +z per site."""
    eu, ev = [], []
    for z in range(lz):
        for y in range(ly):
            for x in range(lx):
                i = (z * ly + y) * lx + x
                if x + 1 < lx:
                    eu.append(i); ev.append(i + 1)
                if y + 1 < ly:
                    eu.append(i); ev.append(i + lx)
                if z + 1 < lz:
                    eu.append(i); ev.append(i + lx * ly)
    m = len(eu)
    return Instance("ising", lx * ly * lz, np.array(eu, np.int32), np.array(ev, np.int32),
                    _pm1(seed, m, 0), None, {"shape": (lx, ly, lz), "seed": seed})


def kings_subgraph(rows: int, cols: int, filling: float, seed: int,
                   weights: str = "unit") -> Instance:
    """King's subgraph: one Bernoulli(filling) draw per grid site row-major
    (site kept iff (x>>11)/2^53 < filling, SplitMix64 stream 0); kept sites are
    renumbered row-major; edges per kept site in directions (0,+1), (+1,-1),
    (+1,0), (+1,+1) (Chebyshev distance 1).  filling >= 1 keeps every site."""
    u = (splitmix64(seed, rows * cols, 0) >> np.uint64(11)).astype(np.float64) / float(1 << 53)
    keep = (u < filling).reshape(rows, cols) if filling < 1.0 else np.ones((rows, cols), bool)
    ids = -np.ones((rows, cols), np.int64)
    ids[keep] = np.arange(int(keep.sum()))
    eu, ev = [], []
    for r in range(rows):
        for c in range(cols):
            if not keep[r, c]:
                continue
            for dr, dc in ((0, 1), (1, -1), (1, 0), (1, 1)):
                rr, cc = r + dr, c + dc
                if 0 <= rr < rows and 0 <= cc < cols and keep[rr, cc]:
                    eu.append(ids[r, c]); ev.append(ids[rr, cc])
    n = int(keep.sum())
    if weights == "unit":
        w = None
    else:  # small integer weights 1..4 (MWIS), stream 1
        w = (1 + (splitmix64(seed, n, 1) >> np.uint64(62)).astype(np.int64)).astype(np.int32)
    pos = np.argwhere(keep)
    return Instance("mis", n, np.array(eu, np.int32).reshape(-1), np.array(ev, np.int32).reshape(-1),
                    None, w, {"shape": (rows, cols), "seed": seed, "keep": keep, "pos": pos})


def column_major_order(inst: "Instance") -> np.ndarray:
    """The kept sites of a King's subgraph (or the sites of a 2-D lattice) column by column: a sweep in the other
    direction than the vertex ids (which are row-major).  Pure geometry; a hint for the library's tree search."""
    if "pos" in inst.meta:
        pos = inst.meta["pos"]
        return np.lexsort((pos[:, 0], pos[:, 1])).astype(np.int32)
    rows, cols = inst.meta["shape"]
    return np.array([r * cols + c for c in range(cols) for r in range(rows)], np.int32)


def random_graph(n: int, p: float, seed: int, kind: str = "ising", field_h: bool = False) -> Instance:
    """Small Erdos-Renyi graph for brute-force pins (edge (i<j) kept iff u < p)."""
    pairs = [(i, j) for i in range(n) for j in range(i + 1, n)]
    u = (splitmix64(seed, len(pairs), 2) >> np.uint64(11)).astype(np.float64) / float(1 << 53)
    sel = [pq for pq, x in zip(pairs, u) if x < p]
    eu = np.array([a for a, _ in sel], np.int32)
    ev = np.array([b for _, b in sel], np.int32)
    if kind == "ising":
        # integer couplings in {-3..3}\{0}, optional integer fields in {-2..2}
        r = splitmix64(seed, len(sel), 3)
        J = ((r % np.uint64(3)).astype(np.int64) + 1) * (2 * ((r >> np.uint64(40)) & np.uint64(1)).astype(np.int64) - 1)
        h = None
        if field_h:
            h = ((splitmix64(seed, n, 4) % np.uint64(5)).astype(np.int64) - 2).astype(np.int32)
        return Instance("ising", n, eu, ev, J.astype(np.int32), h, {"seed": seed})
    w = (1 + (splitmix64(seed, n, 1) % np.uint64(3)).astype(np.int64)).astype(np.int32)
    return Instance("mis", n, eu, ev, None, w, {"seed": seed})


# --------------------------------------------------------------------------
# fixed sets and assignments (Eq. 3: s_{V_f} = x)
# --------------------------------------------------------------------------
def all_assignments(f: int) -> np.ndarray:
    """[2^f][f] uint8, row b holds the bits of b (column j = bit j)."""
    b = np.arange(1 << f, dtype=np.uint32)
    return ((b[:, None] >> np.arange(f, dtype=np.uint32)[None, :]) & 1).astype(np.uint8)


def random_assignments(B: int, f: int, seed: int) -> np.ndarray:
    x = splitmix64(seed, B * max(f, 1), 5) >> np.uint64(63)
    return x.astype(np.uint8).reshape(B, max(f, 1))[:, :f].copy()


def slit_fixed_set_2d(rows: int, cols: int, f: int) -> np.ndarray:
    """f contiguous spins of the middle column, from the top row down: the
    'slit' separator used for config 3 (input recipe)."""
    c = cols // 2
    return np.array([r * cols + c for r in range(f)], np.int32)


def slit_angular_order_2d(rows: int, cols: int, f: int) -> np.ndarray:
    """Elimination order of the free spins of a rows x cols lattice whose slit
    (slit_fixed_set_2d) is fixed: sort by polar angle around the lower end of
    the slit, sweeping from the left leg, under the slit, to the right leg.
    Pure geometry; every ray through the pivot is a vertex separator of
    Chebyshev length, so the contraction width is about max(cols/2, rows-f)+1."""
    c0 = cols // 2
    pr, pc = f - 0.5, float(c0)
    fx = set(int(v) for v in slit_fixed_set_2d(rows, cols, f))
    keyed = []
    for r in range(rows):
        for c in range(cols):
            v = r * cols + c
            if v in fx:
                continue
            # angle measured from the "up" direction, increasing towards the left
            # (counter-clockwise on the page): left leg first, right leg last.
            ang = math.atan2(-(c - pc), -(r - pr))   # up = 0, left = +pi/2
            if ang < 0:
                ang += 2 * math.pi
            if c == c0 and r < f:
                continue
            keyed.append((ang, abs(r - pr) + abs(c - pc), v))
    keyed.sort()
    return np.array([v for _, _, v in keyed], np.int32)


def layer_fixed_set_3d(lx: int, ly: int, lz: int, f: int) -> np.ndarray:
    """f spins of the central z-layer, row-major from its corner (config 4b)."""
    z = lz // 2
    return np.array([(z * ly + (k // lx)) * lx + (k % lx) for k in range(f)], np.int32)


# --------------------------------------------------------------------------
# contraction trees (pure structure; SSA form of include/bbtn.h)
# --------------------------------------------------------------------------
def elimination_tree(index_sets: list[list[int]], order) -> tuple[np.ndarray, np.ndarray]:
    """SSA contraction tree by bucket elimination along a vertex order.

    index_sets[t] = indices carried by input tensor t (ABI order).  For each
    vertex v of `order`, all live tensors carrying v are merged pairwise,
    smallest first (ties: lowest id); leftovers (other components, scalars) are
    merged at the end in id order.  Step t contracts ids (tree_l[t], tree_r[t])
    into id n_inputs + t.  No arithmetic of the method is involved.
    """
    n_in = len(index_sets)
    live: dict[int, frozenset] = {t: frozenset(s) for t, s in enumerate(index_sets)}
    occ: dict[int, set] = {}
    for t, s in live.items():
        for i in s:
            occ.setdefault(i, set()).add(t)
    tl, tr = [], []
    nxt = n_in

    def merge(a: int, b: int) -> int:
        nonlocal nxt
        sa, sb = live.pop(a), live.pop(b)
        for i in sa:
            occ[i].discard(a)
        for i in sb:
            occ[i].discard(b)
        un = sa | sb
        keep = frozenset(i for i in un if len(occ[i]) > 0)   # still carried elsewhere
        live[nxt] = keep
        for i in keep:
            occ[i].add(nxt)
        tl.append(a); tr.append(b)
        nxt += 1
        return nxt - 1

    for v in order:
        v = int(v)
        while True:
            ts = sorted(occ.get(v, ()), key=lambda t: (len(live[t]), t))
            if len(ts) < 2:
                break
            merge(ts[0], ts[1])
    rest = sorted(live.keys(), key=lambda t: (len(live[t]), t))
    while len(rest) > 1:
        c = merge(rest[0], rest[1])
        rest = [c] + rest[2:]
    return np.array(tl, np.int32), np.array(tr, np.int32)


def grouped_elimination_tree(index_sets: list[list[int]], parts) -> tuple[np.ndarray, np.ndarray]:
    """SSA tree that contracts the network PART BY PART and then joins the parts (a divide-and-conquer
    tree, as opposed to the frontier sweep of elimination_tree).

    parts = [(vertex_set, order), ...]: input tensor t belongs to the first part whose vertex_set holds
    every index of t.  Inside a part, bucket elimination along `order` (vertices of the part that occur in
    no other part), then the part's leftover tensors are merged, smallest first, into ONE boundary tensor
    over the vertices the part shares with others.  The part results are then joined left to right in a
    balanced binary fashion: ((P0 P1) (P2 P3)) ...  Pure structure; which index is summed where follows
    from the occurrence rule of the engine and the oracle alike (reading A11)."""
    n_in = len(index_sets)
    owner = [-1] * n_in
    vsets = [set(int(v) for v in vs) for vs, _ in parts]
    for t, s in enumerate(index_sets):
        for p, vs in enumerate(vsets):
            if all(int(i) in vs for i in s):
                owner[t] = p
                break
        assert owner[t] >= 0, f"input tensor {t} fits no part"
    occ_all: dict[int, int] = {}
    for s in index_sets:
        for i in s:
            occ_all[int(i)] = occ_all.get(int(i), 0) + 1
    tl, tr = [], []
    nxt = n_in
    # live[t] = (labels, merged-occurrence counts)
    def merge(live, a, b):
        nonlocal nxt
        (sa, ca), (sb, cb) = live.pop(a), live.pop(b)
        cnt = dict(ca)
        for i, c in cb.items():
            cnt[i] = cnt.get(i, 0) + c
        cnt = {i: c for i, c in cnt.items() if c < occ_all[i]}
        live[nxt] = (frozenset(i for i in (sa | sb) if i in cnt), cnt)
        tl.append(a); tr.append(b)
        nxt += 1
        return nxt - 1
    results = []
    for p, (_, order) in enumerate(parts):
        live = {t: (frozenset(int(i) for i in s), {int(i): 1 for i in s}) for t, s in enumerate(index_sets) if owner[t] == p}
        for v in order:
            v = int(v)
            while True:
                ts = sorted((t for t, (s, _) in live.items() if v in s), key=lambda t: (len(live[t][0]), t))
                if len(ts) < 2:
                    break
                merge(live, ts[0], ts[1])
        while len(live) > 1:
            ts = sorted(live.keys(), key=lambda t: (len(live[t][0]), t))
            merge(live, ts[0], ts[1])
        results.append(live)
    while len(results) > 1:
        nxt_round = []
        for i in range(0, len(results) - 1, 2):
            live = {**results[i], **results[i + 1]}
            a, b = list(results[i].keys())[0], list(results[i + 1].keys())[0]
            merge(live, a, b)
            nxt_round.append(live)
        if len(results) % 2:
            nxt_round.append(results[-1])
        results = nxt_round
    return np.array(tl, np.int32), np.array(tr, np.int32)


def lattice_block_parts(rows: int, cols: int, row_cuts, col_cuts, ids=None, exclude=()):
    """Parts for grouped_elimination_tree on a rows x cols lattice (vertex id r*cols + c, or ids[r][c] with
    -1 for a missing site): rectangular blocks delimited by the separator rows / columns in row_cuts /
    col_cuts; neighbouring blocks SHARE their separator line.  Inside a block the private vertices are
    eliminated row-major.  Vertices in `exclude` (a fixed set) are left out."""
    rb = [0] + list(row_cuts) + [rows - 1]
    cb = [0] + list(col_cuts) + [cols - 1]
    ex = set(int(v) for v in exclude)
    vid = (lambda r, c: r * cols + c) if ids is None else (lambda r, c: int(ids[r][c]))
    blocks = []
    for i in range(len(rb) - 1):
        for j in range(len(cb) - 1):
            blocks.append([vid(r, c) for r in range(rb[i], rb[i + 1] + 1) for c in range(cb[j], cb[j + 1] + 1)
                           if vid(r, c) >= 0 and vid(r, c) not in ex])
    count: dict[int, int] = {}
    for b in blocks:
        for v in b:
            count[v] = count.get(v, 0) + 1
    return [(b, [v for v in b if count[v] == 1]) for b in blocks]


def min_degree_order(inst: "Instance", fixed=()) -> np.ndarray:
    """Greedy min-degree elimination order of the free vertices (ties: fewest fill edges, then lowest
    id) on the graph with `fixed` removed.  Graph structure only."""
    n = inst.n_vertices
    fx = set(int(v) for v in fixed)
    adj = [set() for _ in range(n)]
    for u, v in zip(inst.edge_u, inst.edge_v):
        u, v = int(u), int(v)
        if u in fx or v in fx:
            continue
        adj[u].add(v); adj[v].add(u)
    alive = [v for v in range(n) if v not in fx]
    order = []

    def fill(v):
        nb = list(adj[v])
        return sum(1 for i in range(len(nb)) for j in range(i + 1, len(nb)) if nb[j] not in adj[nb[i]])

    while alive:
        dmin = min(len(adj[x]) for x in alive)
        v = min((x for x in alive if len(adj[x]) == dmin), key=lambda x: (fill(x), x))
        alive.remove(v)
        order.append(v)
        nb = list(adj[v])
        for a in nb:
            adj[a].discard(v)
        for i in range(len(nb)):
            for j in range(i + 1, len(nb)):
                adj[nb[i]].add(nb[j]); adj[nb[j]].add(nb[i])
        adj[v].clear()
    return np.array(order, np.int32)


def tree_fma(index_sets: list[list[int]], tree) -> float:
    """Loop-nest size of a contraction tree: sum over steps of 2^|I_L u I_R| (steps with a rank-0
    operand cost nothing).  A cost model on index sets; no arithmetic of the method."""
    sets = [set(s) for s in index_sets]
    occ: dict[int, int] = {}
    for s in sets:
        for i in s:
            occ[i] = occ.get(i, 0) + 1
    sub = [{i: 1 for i in s} for s in sets]
    live = list(sets)
    fma = 0.0
    for l, r in zip(tree[0], tree[1]):
        l, r = int(l), int(r)
        un = live[l] | live[r]
        cnt = dict(sub[l])
        for i, c in sub[r].items():
            cnt[i] = cnt.get(i, 0) + c
        cnt = {i: c for i, c in cnt.items() if c < occ[i]}
        if live[l] and live[r]:
            fma += float(1 << len(un))
        live.append({i for i in un if i in cnt}); sub.append(cnt)
    return fma


def sequential_tree(n_inputs: int, perm=None) -> tuple[np.ndarray, np.ndarray]:
    """Left-deep chain ((t0 t1) t2) ... in the given input order (a deliberately
    bad but valid tree, used for tree-independence tests on tiny instances)."""
    p = list(range(n_inputs)) if perm is None else [int(x) for x in perm]
    tl, tr = [], []
    cur = p[0]
    for k, t in enumerate(p[1:]):
        tl.append(cur); tr.append(t)
        cur = n_inputs + k
    return np.array(tl, np.int32), np.array(tr, np.int32)


def random_order(n: int, seed: int, exclude=()) -> np.ndarray:
    ex = set(int(v) for v in exclude)
    keys = splitmix64(seed, n, 6)
    order = [int(i) for i in np.argsort(keys, kind="stable") if int(i) not in ex]
    return np.array(order, np.int32)


def natural_order(n: int, exclude=()) -> np.ndarray:
    ex = set(int(v) for v in exclude)
    return np.array([i for i in range(n) if i not in ex], np.int32)


# --------------------------------------------------------------------------
# raw GEMM operands (config 4a) and permutations
# --------------------------------------------------------------------------
def gemm_operands(B: int, M: int, N: int, K: int, seed: int, neg_inf_frac: float = 0.0,
                  wide_counts: bool = False):
    """Energies iid uniform integers in [-64, 64] (x mod 129 - 64), counts iid
    uniform in {1,2,3,4} ((x>>32) mod 4 + 1), SplitMix64 streams 10..13.
    A is [B][M][K], B is [B][K][N], row-major.  With neg_inf_frac > 0 a
    fraction of elements become the zero element (NEG_INF sentinel, count 0);
    wide_counts draws full-range uint64 counts instead (wrap-around test)."""
    def one(shape, s_e, s_c):
        n = int(np.prod(shape))
        x = splitmix64(seed, n, s_e)
        e = ((x % np.uint64(129)).astype(np.int64) - 64).astype(np.int32)
        y = splitmix64(seed, n, s_c)
        if wide_counts:
            c = y.copy()
        else:
            c = ((y >> np.uint64(32)) % np.uint64(4)) + np.uint64(1)
        if neg_inf_frac > 0:
            z = ((x >> np.uint64(20)) & np.uint64(0xFFFF)).astype(np.float64) / 65536.0 < neg_inf_frac
            e[z] = -(1 << 30)
            c[z] = 0
        return e.reshape(shape), c.astype(np.uint64).reshape(shape)
    Ae, Ac = one((B, M, K), 10, 11)
    Be, Bc = one((B, K, N), 12, 13)
    return Ae, Ac, Be, Bc


def random_bit_permutation(r: int, seed: int) -> np.ndarray:
    """perm[j] = source bit that lands on destination bit j (a permutation of 0..r-1)."""
    return np.argsort(splitmix64(seed, r, 7), kind="stable").astype(np.int32)
