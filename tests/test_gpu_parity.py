"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Integer work: the bar is BIT-EXACT for energies and counts."""
import os

import numpy as np
import pytest

from paper_2602_05470_b200 import instances as I

pytestmark = pytest.mark.gpu

NEG_INF = -(1 << 30)
MASK64 = (1 << 64) - 1


@pytest.fixture(scope="module")
def bb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2602_05470_b200 import binding
    binding.load()          # fails loudly if the extension is missing
    return binding


def _to_dev(e, c):
    import torch
    return (torch.from_numpy(np.ascontiguousarray(e)).cuda(),
            torch.from_numpy(np.ascontiguousarray(c).view(np.int64)).cuda())


def _oracle_gemm(oracle, Ae, Ac, Be, Bc):
    Az = (Ae <= -(1 << 29)).astype(np.uint8); Bz = (Be <= -(1 << 29)).astype(np.uint8)
    Ce, Cz, Cc = oracle.gemm(Ae.astype(np.int64), Az, Ac, Be.astype(np.int64), Bz, Bc)
    Ce = np.where(Cz == 1, NEG_INF, Ce).astype(np.int32)
    Cc = np.where(Cz == 1, 0, Cc).astype(np.uint64)
    return Ce, Cc


# ---- K3 alone -------------------------------------------------------------------------
@pytest.mark.parametrize("B,M,N,K,seed,frac,wide", [
    (1, 64, 64, 64, 1, 0.0, False),
    (3, 256, 256, 256, 2, 0.0, False),
    (2, 100, 70, 37, 3, 0.1, False),       # ragged tiles in every dimension + zero elements
    (5, 1, 1, 1, 4, 0.0, False),
    (1, 129, 65, 513, 5, 0.0, True),       # full-range uint64 counts: wrap-around mod 2^64
    (4, 17, 200, 3, 6, 0.5, True),
    (1, 1, 300, 1000, 7, 0.0, False),
    (2, 333, 1, 129, 8, 0.3, False),
    (7, 48, 64, 33, 9, 0.2, False),        # M, N <= 64: the 64x64-tile kernel, ragged, batched
    (3, 64, 37, 70, 10, 0.0, True),
])
def test_gemm_matches_oracle(bb, oracle, B, M, N, K, seed, frac, wide):
    Ae, Ac, Be, Bc = I.gemm_operands(B, M, N, K, seed, neg_inf_frac=frac, wide_counts=wide)
    want_e, want_c = _oracle_gemm(oracle, Ae, Ac, Be, Bc)
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be, Bc)
    # 64: full 64x64 multiply; 32: 32-bit operands, 64-bit accumulators; 3: counts <= 4, 32-bit accumulators;
    # (3, 7): also |energy| < 2^7 promised -> the packed 16x2 form
    # (13, 7) / (32, 7): packed energies with the carry form / with 64-bit accumulators (64x64 tile)
    for bits, ebits in ((64, 32), (32, 32), (14, 32), (3, 32), (3, 7), (13, 7), (32, 7)) if not wide else ((64, 32),):
        Ce, Cc = bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=bits, energy_bits=ebits)
        got_e = Ce.cpu().numpy(); got_c = Cc.cpu().numpy().view(np.uint64)
        assert (got_e == want_e).all(), (bits, ebits)
        assert (got_c == want_c).all(), (bits, ebits)


@pytest.mark.parametrize("B,M,N,K,seed,frac", [
    (2, 256, 256, 512, 41, 0.0),
    (1, 131, 197, 100, 42, 0.2),          # ragged in every dimension, zero elements
    (3, 128, 130, 1000, 43, 0.05),
    (1, 300, 129, 17, 44, 0.5),
])
def test_gemm_packed_form_full_energy_range(bb, oracle, B, M, N, K, seed, frac):
    # the packed 16x2 form (energy_bits <= 11, 32-bit accumulators) on energies that use its whole range
    # (-2047..2047, ties made frequent by drawing from a few hundred values) and on the zero element
    Ae, Ac, Be, Bc = I.gemm_operands(B, M, N, K, seed, neg_inf_frac=frac)
    spread = lambda e, s: np.where(e <= -(1 << 29), e, ((e.astype(np.int64) * 31 + s) % 4095 - 2047)).astype(np.int32)
    Ae, Be = spread(Ae, 7), spread(Be, 1900)
    assert Ae.max() > 1900 and Be[Be > -(1 << 29)].min() < -1900
    want_e, want_c = _oracle_gemm(oracle, Ae, Ac, Be, Bc)
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be, Bc)
    prev = bb.set_debug_checks(True)
    try:
        for ebits, bits in ((11, 3), (32, 3), (11, 13), (11, 32)):       # 32-bit, carry-form and 64-bit accumulators
            Ce, Cc = bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=bits, energy_bits=ebits)
            assert (Ce.cpu().numpy() == want_e).all(), (ebits, bits)
            assert (Cc.cpu().numpy().view(np.uint64) == want_c).all(), (ebits, bits)
        with pytest.raises(bb.BbtnError):                              # |e| up to 2047 is not below 2^10
            bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=3, energy_bits=10)
    finally:
        bb.set_debug_checks(prev)


def test_gemm_narrow_counts_long_sums(bb, oracle):
    # count_bits = 14: chunk-local 32-bit tie sums added to 64-bit accumulators; all energies equal, so every term ties
    # and the totals (up to 2000 * 2^28) need the 64 bits
    B, M, N, K = 2, 130, 70, 2000
    Ae, Ac, Be, Bc = I.gemm_operands(B, M, N, K, seed=51)
    Ae[:] = 3; Be[:] = -5
    Ac = (I.splitmix64(51, Ac.size, 30) % np.uint64(1 << 14)).reshape(Ac.shape)
    Bc = (I.splitmix64(51, Bc.size, 31) % np.uint64(1 << 14)).reshape(Bc.shape)
    want_e, want_c = _oracle_gemm(oracle, Ae, Ac, Be, Bc)
    assert int(want_c.max()) > 1 << 36
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be, Bc)
    for bits in (14, 32, 64):
        Ce, Cc = bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=bits)
        assert (Ce.cpu().numpy() == want_e).all() and (Cc.cpu().numpy().view(np.uint64) == want_c).all(), bits


@pytest.mark.parametrize("bits,kmod", [(13, 1), (13, 3), (32, 1), (32, 5), (20, 2)])
def test_gemm_packed_form_wide_counts_long_tie_sums(bb, oracle, bits, kmod):
    # the packed form beyond 32-bit totals: the carry form (operand counts < 2^13: bit 31 of the running sum moves into
    # a second register after every chunk) and 64-bit accumulators (operand counts < 2^32, totals wrap mod 2^64).
    # Energies take kmod distinct values per operand so that a large share of the K terms tie (kmod = 1: all of them),
    # and the maximum keeps rising along k for kmod > 1 (resets of both accumulator halves)
    B, M, N, K = 2, 130, 70, 1500
    Ae, Ac, Be, Bc = I.gemm_operands(B, M, N, K, seed=300 + bits + kmod, neg_inf_frac=0.02 if kmod > 1 else 0.0)
    fin_a, fin_b = Ae > -(1 << 29), Be > -(1 << 29)
    ramp_a = (np.arange(K)[None, None, :] * kmod // K).astype(np.int32)           # rises along k: later chunks beat earlier ones
    Ae = np.where(fin_a, (Ae % kmod) + ramp_a, Ae).astype(np.int32)
    Be = np.where(fin_b, Be % kmod, Be).astype(np.int32)
    Ac = np.where(fin_a, I.splitmix64(7, Ac.size, 40).reshape(Ac.shape) % np.uint64(1 << bits), 0).astype(np.uint64)
    Bc = np.where(fin_b, I.splitmix64(7, Bc.size, 41).reshape(Bc.shape) % np.uint64(1 << bits), 0).astype(np.uint64)
    want_e, want_c = _oracle_gemm(oracle, Ae, Ac, Be, Bc)
    if bits == 13 and kmod == 1:
        assert int(want_c.max()) > 1 << 33                                      # carries out of bit 31 happened
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be, Bc)
    prev = bb.set_debug_checks(True)
    try:
        for cb, eb in ((bits, 7), (bits, 32), (64, 32)):
            Ce, Cc = bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=cb, energy_bits=eb)
            assert (Ce.cpu().numpy() == want_e).all(), (cb, eb)
            assert (Cc.cpu().numpy().view(np.uint64) == want_c).all(), (cb, eb)
    finally:
        bb.set_debug_checks(prev)


def test_gemm_shared_operand_stride0(bb, oracle):
    Ae, Ac, Be, Bc = I.gemm_operands(4, 96, 80, 72, seed=11)
    want_e, want_c = _oracle_gemm(oracle, Ae, Ac, np.broadcast_to(Be[0], Be.shape).copy(), np.broadcast_to(Bc[0], Bc.shape).copy())
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be[0], Bc[0])
    Ce, Cc = bb.tropical_gemm_batched(dAe, dAc, dBe, dBc)
    assert (Ce.cpu().numpy() == want_e).all() and (Cc.cpu().numpy().view(np.uint64) == want_c).all()


def test_gemm_4096_sampled_rows_all_count_modes(bb, oracle):
    # BASELINE config 4a's largest size: 64 sampled full rows (SURVEY 8(c) pin vi) in the three count modes
    n = 4096
    Ae, Ac, Be, Bc = I.gemm_operands(1, n, n, n, seed=31)
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be, Bc)
    rows = np.unique((I.splitmix64(7, 64, 20) % np.uint64(n)).astype(np.int64))
    we, wc = _oracle_gemm(oracle, Ae[:, rows], Ac[:, rows], Be, Bc)
    for bits, ebits in ((64, 32), (32, 32), (14, 32), (3, 32), (3, 7)):
        Ce, Cc = bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=bits, energy_bits=ebits)
        got_e = Ce[0].cpu().numpy(); got_c = Cc[0].cpu().numpy().view(np.uint64)
        assert (got_e[rows] == we[0]).all() and (got_c[rows] == wc[0]).all(), (bits, ebits)
        # cheap whole-matrix property: every output energy is attainable (<= 128) and every count is in [1, 16 n]
        assert got_e.max() <= 128 and got_e.min() >= 100 and got_c.min() >= 1 and got_c.max() <= 16 * n


def test_debug_checks_catch_a_broken_promise(bb):
    # count_bits is a caller promise (include/bbtn.h); with bbtn_set_debug_checks the device verifies it
    Ae, Ac, Be, Bc = I.gemm_operands(2, 96, 80, 72, seed=12)
    Ac = Ac.copy(); Ac[1, 5, 7] = 70000
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be, Bc)
    prev = bb.set_debug_checks(True)
    try:
        bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=17)            # 70000 < 2^17: fine
        with pytest.raises(bb.BbtnError) as e:
            bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=3)
        assert e.value.status == bb.BBTN_EINVAL and "count" in str(e.value)
        Be2 = Be.copy(); Be2[0, 3, 3] = -(1 << 29) - 1                         # a non-canonical zero element
        dBe2, _ = _to_dev(Be2, Bc)
        with pytest.raises(bb.BbtnError) as e:
            bb.tropical_gemm_batched(dAe, dAc, dBe2, dBc, count_bits=64)
        assert e.value.status == bb.BBTN_EINVAL and "energy" in str(e.value)
        with pytest.raises(bb.BbtnError):
            bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=0)
    finally:
        bb.set_debug_checks(prev)


def test_gemm_large_sampled_rows(bb, oracle):
    # BASELINE config 4a size n = 1024: full oracle is 1e9 FMAs; check 16 sampled rows of one batch entry
    n, B = 1024, 2
    Ae, Ac, Be, Bc = I.gemm_operands(B, n, n, n, seed=21)
    dAe, dAc = _to_dev(Ae, Ac); dBe, dBc = _to_dev(Be, Bc)
    rows = (I.splitmix64(5, 16, 20) % np.uint64(n)).astype(np.int64)
    want = [_oracle_gemm(oracle, Ae[b:b + 1, rows], Ac[b:b + 1, rows], Be[b:b + 1], Bc[b:b + 1]) for b in range(B)]
    for bits, ebits in ((64, 32), (32, 32), (3, 32), (3, 7)):      # (3, 7) is the launch configuration bench.py times
        Ce, Cc = bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, count_bits=bits, energy_bits=ebits)
        got_e = Ce.cpu().numpy(); got_c = Cc.cpu().numpy().view(np.uint64)
        for b in range(B):
            we, wc = want[b]
            assert (got_e[b, rows] == we[0]).all() and (got_c[b, rows] == wc[0]).all()


# ---- K2 alone -------------------------------------------------------------------------
@pytest.mark.parametrize("r,B,seed", [(0, 3, 0), (1, 2, 1), (3, 5, 2), (7, 3, 3), (12, 4, 4), (16, 2, 5), (20, 1, 6)])
def test_permute_matches_oracle(bb, oracle, r, B, seed):
    n = 1 << r
    perm = I.random_bit_permutation(r, seed)
    src_e = (I.splitmix64(seed, B * n, 8) % np.uint64(100000)).astype(np.int32).reshape(B, n)
    src_c = I.splitmix64(seed, B * n, 9).reshape(B, n)
    want_e, want_c = oracle.permute(perm, src_e, src_c)
    de, dc = _to_dev(src_e, src_c)
    oe, oc = bb.permute_batched(perm, de, dc)
    assert (oe.cpu().numpy() == want_e).all() and (oc.cpu().numpy().view(np.uint64) == want_c).all()
    # pi then pi^-1 is the identity
    be_, bc_ = bb.permute_batched(np.argsort(perm).astype(np.int32), oe, oc)
    assert (be_.cpu().numpy() == src_e).all() and (bc_.cpu().numpy().view(np.uint64) == src_c).all()


def test_permute_structured(bb, oracle):
    # identity, full reversal, a single high<->low swap and a rotation (typical "move k to the top")
    r, B = 14, 2
    n = 1 << r
    src_e = (I.splitmix64(1, B * n, 8) % np.uint64(1000)).astype(np.int32).reshape(B, n)
    src_c = I.splitmix64(1, B * n, 9).reshape(B, n)
    de, dc = _to_dev(src_e, src_c)
    ident = np.arange(r, dtype=np.int32)
    swap = ident.copy(); swap[0], swap[r - 1] = swap[r - 1], swap[0]
    for perm in (ident, ident[::-1].copy(), swap, np.roll(ident, 3), np.roll(ident, -1)):
        want_e, want_c = oracle.permute(perm, src_e, src_c)
        oe, oc = bb.permute_batched(perm, de, dc)
        assert (oe.cpu().numpy() == want_e).all() and (oc.cpu().numpy().view(np.uint64) == want_c).all()


# ---- whole path: K1 -> (K2) -> K3 -> K4 -----------------------------------------------
# auto / streaming run small networks as ONE launch (one CTA per leaf, tensors in shared memory); the *_nofused modes
# keep the per-node kernels (K1, streaming K3, K4) covered on the same instances
MODES = {"auto": 0, "streaming": 0x10, "tiled": 0x20, "auto_nograph": 0x4, "nofused": 0x80, "streaming_nofused": 0x90,
         "nofused_nograph": 0x84}


def _check_leaves(bb, oracle, inst, tree, fixed, assign, flags=0, sample=None):
    h = bb.Handle(inst, tree=tree, flags=flags)
    energy, count = h.contract_batch(fixed, assign)[:2]
    idx = range(len(assign)) if sample is None else sample
    for b in idx:
        we, wc = oracle.contract_tree(inst, tree[0], tree[1], fixed, assign[b]) if tree is not None else \
            oracle.frontier_dp(inst, None, fixed, assign[b])
        if we is None:
            assert energy[b] == NEG_INF and count[b] == 0
        else:
            assert int(energy[b]) == we, (b, energy[b], we)
            assert int(count[b]) == wc & MASK64, (b, count[b], wc)
    h.close()
    return energy, count


@pytest.mark.parametrize("seed", range(1, 11))
def test_config1_ising_6x6_unbranched(bb, oracle, seed):
    # BASELINE config 1: 6x6 open +-J, 36 spins / 60 bonds, no field, no branching
    inst = I.ising_lattice_2d(6, 6, seed)
    assert inst.n_vertices == 36 and inst.n_edges == 60
    tree = I.elimination_tree(inst.input_index_sets(), I.natural_order(36))
    want = oracle.contract_tree(inst, *tree)
    assert want == oracle.frontier_dp(inst)
    for mode, fl in MODES.items():
        h = bb.Handle(inst, tree=tree, flags=fl)
        e, c = h.contract_batch()
        assert (int(e[0]), int(c[0])) == want, mode
    h = bb.Handle(inst)                  # library-derived tree
    e, c = h.contract_batch()
    assert (int(e[0]), int(c[0])) == want


@pytest.mark.parametrize("seed", range(1, 11))
def test_config2_kings_12x12(bb, oracle, seed):
    # BASELINE config 2: King's subgraph 12x12, filling 0.8, unit weights
    k = I.kings_subgraph(12, 12, 0.8, seed)
    tree = I.elimination_tree(k.input_index_sets(), I.natural_order(k.n_vertices))
    want = oracle.contract_tree(k, *tree)
    assert want == oracle.frontier_dp(k)
    for mode, fl in MODES.items():
        h = bb.Handle(k, tree=tree, flags=fl)
        e, c = h.contract_batch()
        assert (int(e[0]), int(c[0])) == want, mode


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("case", range(6))
def test_sliced_batches_all_modes(bb, oracle, mode, case):
    if case == 0:
        inst = I.ising_lattice_2d(5, 6, 3, field_h=1)
    elif case == 1:
        inst = I.kings_subgraph(6, 6, 0.8, 4, weights="rand")
    elif case == 2:
        inst = I.ising_lattice_3d(3, 3, 3, 5)
    elif case == 3:
        inst = I.random_graph(18, 0.25, 6, "ising", field_h=True)
    elif case == 4:
        inst = I.random_graph(20, 0.2, 7, "mis")
    else:
        inst = I.kings_subgraph(7, 5, 0.6, 8)            # isolated vertices likely (reading A7)
    n = inst.n_vertices
    f = 4
    fixed = I.random_order(n, 40 + case)[:f]
    assign = I.all_assignments(f)
    # one tree built on the sliced network, one on the unsliced network (rank-0 inputs stay in the tree)
    t_sliced = I.elimination_tree(inst.input_index_sets(fixed), I.random_order(n, 60 + case, exclude=fixed))
    t_full = I.elimination_tree(inst.input_index_sets(), I.natural_order(n))
    for tree in (t_sliced, t_full):
        e, c = _check_leaves(bb, oracle, inst, tree, fixed, assign, MODES[mode])
    # Eq. 3: (+) over all leaves == unbranched
    whole = oracle.contract_tree(inst, *t_full)
    feas = e != NEG_INF
    if inst.kind == "ising":
        best = int(e[feas].min())
    else:
        best = int(e[feas].max())
    tot = sum(int(x) for x in c[feas & (e == best)])
    assert (best, tot & MASK64) == (whole[0], whole[1] & MASK64)


def test_infeasible_leaves_and_empty_fixed(bb, oracle):
    k = I.kings_subgraph(4, 4, 1.0, 1)
    fixed = np.array([0, 1, 5], np.int32)
    assign = I.all_assignments(3)
    tree = I.elimination_tree(k.input_index_sets(), I.natural_order(16))
    e, c = _check_leaves(bb, oracle, k, tree, fixed, assign)
    assert (e == NEG_INF).sum() == 4 and (c[e == NEG_INF] == 0).all()   # any two of {0,1,5} both in: adjacent
    # everything fixed: the network is all scalars
    inst = I.ising_lattice_2d(2, 3, 2, field_h=1)
    fixed = np.arange(6, dtype=np.int32)
    assign = I.all_assignments(6)
    h = bb.Handle(inst)
    e, c = h.contract_batch(fixed, assign)
    for b in range(64):
        we, wc = oracle.exhaustive(inst, fixed, assign[b])
        assert (int(e[b]), int(c[b])) == (we, wc)


def test_counts_wrap_mod_2_64_and_crt(bb, oracle):
    # 30 disjoint AF triangles: count 6^30 > 2^64; 70 isolated spins: 2^70
    import itertools
    edges = []
    for t in range(30):
        edges += [(3 * t, 3 * t + 1), (3 * t + 1, 3 * t + 2), (3 * t, 3 * t + 2)]
    n = 90 + 70
    inst = I.Instance("ising", n, np.array([a for a, _ in edges], np.int32), np.array([b for _, b in edges], np.int32),
                      -np.ones(len(edges), np.int32), None)
    true = 6 ** 30 * 2 ** 70
    h = bb.Handle(inst, flags=bb.BBTN_COUNT_CRT)
    e, c, cm = h.contract_batch()
    assert int(e[0]) == -30
    assert int(c[0]) == true % (1 << 64)
    assert int(cm[0, 0]) == true % bb.BBTN_P1 and int(cm[0, 1]) == true % bb.BBTN_P2
    # CRT recovers counts below 2^64 * P1 * P2 ~ 2^126
    inst2 = I.Instance("ising", 90, inst.edge_u, inst.edge_v, inst.edge_w, None)
    h2 = bb.Handle(inst2, flags=bb.BBTN_COUNT_CRT)
    e, c, cm = h2.contract_batch()
    assert bb.crt_combine(c[0], cm[0, 0], cm[0, 1]) == 6 ** 30
    # CRT residues on a branched lattice batch agree with the oracle's big integers
    lat = I.ising_lattice_2d(6, 6, 9)
    fixed = np.array([14, 15, 20], np.int32); assign = I.all_assignments(3)
    tree = I.elimination_tree(lat.input_index_sets(fixed), I.natural_order(36, exclude=fixed))
    h3 = bb.Handle(lat, tree=tree, flags=bb.BBTN_COUNT_CRT)
    e, c, cm = h3.contract_batch(fixed, assign)
    for b in range(8):
        we, wc = oracle.contract_tree(lat, tree[0], tree[1], fixed, assign[b])
        assert int(e[b]) == we and int(c[b]) == wc % (1 << 64)
        assert int(cm[b, 0]) == wc % bb.BBTN_P1 and int(cm[b, 1]) == wc % bb.BBTN_P2


def test_closed_forms_on_gpu(bb):
    # north_star closed forms, straight through the CUDA path
    for L in (3, 8, 12):
        inst = I.ising_lattice_2d(L, L, 1, ferro=True)
        e, c = bb.Handle(inst, tree=I.elimination_tree(inst.input_index_sets(), I.natural_order(L * L))).contract_batch()
        assert (int(e[0]), int(c[0])) == (-2 * L * (L - 1), 2)
    for L in (3, 5, 7, 9):
        k = I.kings_subgraph(L, L, 1.0, 1)
        e, c = bb.Handle(k, tree=I.elimination_tree(k.input_index_sets(), I.natural_order(L * L))).contract_batch()
        assert (int(e[0]), int(c[0])) == (((L + 1) // 2) ** 2, 1)


def test_config3_shape_branched_lattice_sampled(bb, oracle):
    # config 3 at reduced size (12x12, slit of 6 -> 64 leaves): every leaf vs oracle-2, leaf-sum vs oracle-3
    L, f = 12, 6
    inst = I.ising_lattice_2d(L, L, 5)
    fixed = I.slit_fixed_set_2d(L, L, f)
    tree = I.elimination_tree(inst.input_index_sets(fixed), I.slit_angular_order_2d(L, L, f))
    assign = I.all_assignments(f)
    e, c = _check_leaves(bb, oracle, inst, tree, fixed, assign, sample=range(0, 64, 7))
    whole = oracle.frontier_dp(inst)
    best = int(e.min())
    assert (best, sum(int(x) for x in c[e == best]) & MASK64) == (whole[0], whole[1] & MASK64)


# ---- divide-and-conquer trees: the joins run K2 + tiled K3 (automatic mode) and the long-reduction kernel ----
def _king_ids(k, rows, cols):
    ids = -np.ones((rows, cols), int)
    ids[k.meta["keep"]] = np.arange(k.n_vertices)
    return ids


@pytest.mark.parametrize("case", ["ising12", "ising16", "king12", "ising12-sliced", "king12-sliced"])
def test_block_tree_runs_tiled_gemm_and_trace_kernels(bb, oracle, case):
    # four blocks contracted to boundary tensors, then joined: (TL x TR) and (BL x BR) are permute + tiled GEMM
    # nodes in AUTOMATIC mode (>= 4 summed, >= 5 free indices on both sides), the last join is a 2^k-term trace
    if case.startswith("ising"):
        L = 16 if "16" in case else 12
        inst = I.ising_lattice_2d(L, L, 3 if L == 12 else 4)
        ids = None
    else:
        L = 12
        inst = I.kings_subgraph(L, L, 1.0, 6, weights="rand")
        ids = _king_ids(inst, L, L)
    fixed, assign = None, None
    if case.endswith("sliced"):
        v = lambda r, c: r * L + c if ids is None else int(ids[r][c])
        fixed = np.array([v(2, 2), v(2, L - 3), v(L - 3, 3)], np.int32)        # one private vertex in three of the blocks
        assign = I.all_assignments(3)
    parts = I.lattice_block_parts(L, L, [L // 2], [L // 2], ids, exclude=() if fixed is None else fixed)
    tree = I.grouped_elimination_tree(inst.input_index_sets(() if fixed is None else fixed), parts)
    h = bb.Handle(inst, tree=tree, flags=bb.BBTN_COUNT_CRT)
    info = h.plan_query(fixed, 1 if assign is None else len(assign))
    assert info["n_gemm_tiled"] > 0 and info["n_permute"] > 0 and info["n_trace"] > 0, info
    energy, count, cmod = h.contract_batch(fixed, assign)
    for b in range(len(energy)):
        we, wc = oracle.contract_tree(inst, tree[0], tree[1], fixed, None if assign is None else assign[b])
        assert (int(energy[b]), int(count[b])) == (we, wc & MASK64), (case, b)
        assert (int(cmod[b, 0]), int(cmod[b, 1])) == (wc % bb.BBTN_P1, wc % bb.BBTN_P2), (case, b)
    h.close()
    if fixed is None:
        assert (we, wc) == oracle.frontier_dp(inst)


@pytest.mark.parametrize("mode", ["auto", "streaming"])
def test_join_over_13_summed_indices(bb, oracle, mode):
    # three column blocks of a 13-row lattice: the first join sums the 13 spins of a separator column into a
    # rank-13 output (streaming K3 with a 2^13-term sum per output: more than 12 summed indices), the last join
    # is a 13-index trace
    inst = I.ising_lattice_2d(13, 7, 5)
    parts = I.lattice_block_parts(13, 7, [], [2, 4])
    tree = I.grouped_elimination_tree(inst.input_index_sets(), parts)
    want = oracle.contract_tree(inst, *tree)
    assert want == oracle.frontier_dp(inst)
    h = bb.Handle(inst, tree=tree, flags=MODES[mode] | bb.BBTN_COUNT_CRT)
    info = h.plan_query()
    assert info["n_trace"] >= 1 and info["max_rank"] == 26
    e, c, cm = h.contract_batch()
    assert (int(e[0]), int(c[0])) == (want[0], want[1] & MASK64)
    assert (int(cm[0, 0]), int(cm[0, 1])) == (want[1] % bb.BBTN_P1, want[1] % bb.BBTN_P2)
    h.close()


@pytest.mark.parametrize("rows,cols,cuts", [(8, 3, [1]), (9, 4, [1, 2]), (7, 5, [2])])
def test_tree_gemm_with_small_counts_takes_the_packed_kmajor_form(bb, oracle, rows, cols, cuts):
    # FORCE_TILED on thin column blocks: the joins are GEMMs with M = 2^rows (> 64) whose operands have summed only a
    # few vertices, so the planner's count bound allows 32-bit accumulators and the problem's energy bound the packed
    # 16x2 form -- the k-major (engine-layout) instantiation of gemm_pack16_kernel, which the raw ABI never reaches
    inst = I.ising_lattice_2d(rows, cols, 11 + rows, field_h=1)
    tree = I.grouped_elimination_tree(inst.input_index_sets(), I.lattice_block_parts(rows, cols, [], cuts))
    want = oracle.contract_tree(inst, *tree)
    assert want == oracle.frontier_dp(inst)
    for flags in (bb.BBTN_FORCE_TILED, bb.BBTN_FORCE_TILED | bb.BBTN_COUNT_CRT):
        h = bb.Handle(inst, tree=tree, flags=flags)
        assert h.plan_query()["n_gemm_tiled"] > 0
        out = h.contract_batch()
        assert (int(out[0][0]), int(out[1][0])) == (want[0], want[1] & MASK64)
        h.close()
    # the same with a sliced batch (leaf-variant operands: batch strides on A or B)
    fixed = np.array([0, rows * cols - 1], np.int32)
    parts = I.lattice_block_parts(rows, cols, [], cuts, exclude=fixed)
    t2 = I.grouped_elimination_tree(inst.input_index_sets(fixed), parts)
    _check_leaves(bb, oracle, inst, t2, fixed, I.all_assignments(2), bb.BBTN_FORCE_TILED)


def test_batch_size_and_order_independence(bb):
    inst = I.ising_lattice_2d(8, 8, 3)
    fixed = I.slit_fixed_set_2d(8, 8, 4)
    tree = I.elimination_tree(inst.input_index_sets(fixed), I.slit_angular_order_2d(8, 8, 4))
    assign = I.all_assignments(4)
    h = bb.Handle(inst, tree=tree)
    e_all, c_all = h.contract_batch(fixed, assign)
    for b in (0, 5, 15):
        e1, c1 = h.contract_batch(fixed, assign[b:b + 1])
        assert e1[0] == e_all[b] and c1[0] == c_all[b]
    perm = np.argsort(I.splitmix64(1, 16, 0))
    e_p, c_p = h.contract_batch(fixed, assign[perm])
    assert (e_p == e_all[perm]).all() and (c_p == c_all[perm]).all()


# ---- K5 + host B&B ---------------------------------------------------------------------
def _grid_regions(rows, cols, br, bc, ids=None):
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


@pytest.mark.parametrize("case", range(4))
def test_region_bound_matches_oracle(bb, oracle, case):
    rows, cols = 6, 7
    if case % 2 == 0:
        inst = I.ising_lattice_2d(rows, cols, case, field_h=case - 1)
        ids = None
    else:
        inst = I.kings_subgraph(rows, cols, 0.8, case, weights="rand" if case == 3 else "unit")
        ids = -np.ones((rows, cols), int); ids[inst.meta["keep"]] = np.arange(inst.n_vertices)
    offs, verts = _grid_regions(rows, cols, 3, 3, ids)
    f = 5
    fixed = I.random_order(inst.n_vertices, 90 + case)[:f]
    assign = I.all_assignments(f)
    h = bb.Handle(inst)
    got = h.region_bound(offs, verts, fixed, assign)
    energy, _ = h.contract_batch(fixed, assign)
    for b in range(len(assign)):
        want = oracle.region_bound(inst, offs, verts, fixed, assign[b])
        if want is None:
            assert got[b] == NEG_INF
            continue
        assert int(got[b]) == (-want if inst.kind == "ising" else want)
        # admissible: never cuts off the exact value of the leaf
        if inst.kind == "ising":
            assert got[b] <= energy[b]
        else:
            assert got[b] >= energy[b]
    # no regions at all, and no fixed vertices
    got0 = h.region_bound([0], [], fixed, assign)
    for b in (0, 7, 31):
        want = oracle.region_bound(inst, [0], [], fixed, assign[b])
        assert (got0[b] == NEG_INF) if want is None else int(got0[b]) == (-want if inst.kind == "ising" else want)
    w = oracle.region_bound(inst, offs, verts)
    assert int(h.region_bound(offs, verts)[0]) == (-w if inst.kind == "ising" else w)


@pytest.mark.parametrize("case", range(4))
def test_solve_bb_matches_unbranched(bb, oracle, case):
    if case % 2 == 0:
        rows, cols = 8, 8
        inst = I.ising_lattice_2d(rows, cols, 10 + case)
        ids = None
        branch = np.array([r * cols + cols // 2 for r in range(rows)], np.int32)
    else:
        rows, cols = 9, 9
        inst = I.kings_subgraph(rows, cols, 0.8, 10 + case)
        ids = -np.ones((rows, cols), int); ids[inst.meta["keep"]] = np.arange(inst.n_vertices)
        branch = np.array([ids[r][cols // 2] for r in range(rows) if ids[r][cols // 2] >= 0], np.int32)
    offs, verts = _grid_regions(rows, cols, 3, 3, ids)
    whole = oracle.frontier_dp(inst)
    h = bb.Handle(inst, flags=bb.BBTN_COUNT_CRT)
    for pruning in (False, True):
        out = h.solve_bb(branch, 3, offs, verts, max_batch=64, use_pruning=pruning)
        assert (out["energy"], out["count"]) == (whole[0], whole[1] & MASK64)
        assert out["count_mod"] == (whole[1] % bb.BBTN_P1, whole[1] % bb.BBTN_P2)
        if not pruning and inst.kind == "ising":
            assert out["contracted"] == 1 << len(branch)
    assert out["contracted"] <= 1 << len(branch)


# ---- BASELINE configs at FULL size vs goldens written by the oracle (tests/golden/make_config_goldens.py) ----
def _goldens():
    import json
    with open(os.path.join(os.path.dirname(__file__), "golden", "config_goldens.json")) as f:
        return json.load(f)["cases"]


def _expect(name):
    g = _goldens()[name]
    return int(g["energy"]), int(g["count"]) & MASK64


def _sampled_leaves(B, n, seed):
    return sorted(set(int(x) for x in (I.splitmix64(seed, n, 21) % np.uint64(B))) | {0, B - 1})


@pytest.mark.parametrize("f", [8, 10, 12])
def test_config3_full_size_leaf_by_leaf(bb, oracle, f):
    # BASELINE config 3 at full size in the launch configuration that is timed (all 2^f leaves, one call):
    # 16 seeded leaves + the first and the last compared ONE BY ONE with the oracle's naive contraction of the same tree
    inst = I.ising_lattice_2d(24, 24, 1)
    fixed = I.slit_fixed_set_2d(24, 24, f)
    tree = I.elimination_tree(inst.input_index_sets(fixed), I.slit_angular_order_2d(24, 24, f))
    assign = I.all_assignments(f)
    h = bb.Handle(inst, tree=tree, max_elements_per_leaf=1 << 26)
    energy, count = h.contract_batch(fixed, assign)
    h.close()
    for b in _sampled_leaves(1 << f, 16, 100 + f):
        we, wc = oracle.contract_tree(inst, tree[0], tree[1], fixed, assign[b])
        assert (int(energy[b]), int(count[b])) == (we, wc & MASK64), (f, b)
    assert bb.oplus_combine("ising", energy, count)[:2] == _expect("config3 ising 24x24 seed 1")


@pytest.mark.parametrize("f", [6, 8, 10])
def test_config4b_full_size_leaf_by_leaf(bb, oracle, f):
    inst = I.ising_lattice_3d(5, 5, 5, 1)
    fixed = I.layer_fixed_set_3d(5, 5, 5, f)
    tree = I.elimination_tree(inst.input_index_sets(fixed), I.min_degree_order(inst, fixed))
    assign = I.all_assignments(f)
    h = bb.Handle(inst, tree=tree, max_elements_per_leaf=1 << 26)
    energy, count = h.contract_batch(fixed, assign)
    h.close()
    for b in _sampled_leaves(1 << f, 3 if f == 6 else 16, 200 + f):
        we, wc = oracle.contract_tree(inst, tree[0], tree[1], fixed, assign[b])
        assert (int(energy[b]), int(count[b])) == (we, wc & MASK64), (f, b)
    assert bb.oplus_combine("ising", energy, count)[:2] == _expect("config4b ising 5x5x5 seed 1")


@pytest.mark.parametrize("case", ["cube-crt", "ising24-crt", "king16-crt", "cube-search", "ising14-tiled"])
def test_small_subtrees_run_as_shared_memory_prologue(bb, oracle, case):
    # larger plans run their small subtrees (every tensor <= 2^12 elements) as one or two shared-memory launches and only
    # the rest of the tree node by node (api.cu prepare_hybrid): far fewer launches than tree nodes, the same integers
    # as the per-node form (BBTN_NO_FUSED) on every leaf, and the oracle's on sampled leaves -- all three count rings
    if case.startswith("cube"):
        inst = I.ising_lattice_3d(4, 4, 5, 2); f = 4
        fixed = I.layer_fixed_set_3d(4, 4, 5, f)
        tree = I.elimination_tree(inst.input_index_sets(fixed), I.min_degree_order(inst, fixed))
    elif case.startswith("ising24"):
        inst = I.ising_lattice_2d(24, 24, 5, field_h=1); f = 8
        fixed = I.slit_fixed_set_2d(24, 24, f)
        tree = I.elimination_tree(inst.input_index_sets(fixed), I.slit_angular_order_2d(24, 24, f))
    elif case.startswith("king16"):
        inst = I.kings_subgraph(16, 16, 0.8, 3, weights="rand"); f = 5
        ids = _king_ids(inst, 16, 16)
        fixed = np.array([ids[r][8] for r in range(16) if ids[r][8] >= 0][:f], np.int32)
        tree = None
    else:
        inst = I.ising_lattice_2d(14, 14, 6); f = 3
        ids = None
        fixed = np.array([2 * 14 + 2, 2 * 14 + 11, 11 * 14 + 3], np.int32)
        parts = I.lattice_block_parts(14, 14, [7], [7], None, exclude=fixed)
        tree = I.grouped_elimination_tree(inst.input_index_sets(fixed), parts)
    assign = I.all_assignments(len(fixed))
    search = case.endswith("search")
    base = bb.BBTN_SEARCH_ONLY if search else (bb.BBTN_COUNT_CRT if case.endswith("crt") else 0)
    h = bb.Handle(inst, tree=tree, flags=base)
    info = h.plan_query(fixed, len(assign))
    assert info["n_kernel_launches"] < info["n_nodes"] // 2, info       # the prologue is active
    got = h.contract_batch(fixed, assign)
    got2 = h.contract_batch(fixed, assign[::-1].copy())                   # again (CUDA graph replay), other leaves
    h.close()
    h0 = bb.Handle(inst, tree=tree, flags=base | bb.BBTN_NO_FUSED)
    info0 = h0.plan_query(fixed, len(assign))
    assert info0["n_kernel_launches"] > info0["n_nodes"]
    ref = h0.contract_batch(fixed, assign)
    h0.close()
    for x, y in zip(got, ref):
        assert (x == y).all(), case
    for x, y in zip(got2, ref):
        assert (x == y[::-1]).all(), case
    tl, tr = tree if tree is not None else (None, None)
    for b in _sampled_leaves(len(assign), 6, 17):
        if tree is not None:
            we, wc = oracle.contract_tree(inst, tl, tr, fixed, assign[b])
        else:
            we, wc = oracle.frontier_dp(inst, None, fixed, assign[b])
            we = NEG_INF if we is None else we
        assert int(got[0][b]) == we, (case, b)
        if not search:
            assert int(got[1][b]) == wc & MASK64, (case, b)
            if case.endswith("crt"):
                assert (int(got[2][b, 0]), int(got[2][b, 1])) == (wc % bb.BBTN_P1, wc % bb.BBTN_P2), (case, b)


def test_config3_full_size_24x24_all_leaves(bb):
    # the launch configuration time_to_solve.py times: slit of f spins, all 2^f leaves in one call
    from paper_2602_05470_b200 import time_to_solve as T
    inst = I.ising_lattice_2d(24, 24, 1)
    for f in (8, 10, 12):
        fixed = I.slit_fixed_set_2d(24, 24, f)
        tree = I.elimination_tree(inst.input_index_sets(fixed), I.slit_angular_order_2d(24, 24, f))
        out = T.solve_branched("config3", inst, fixed, tree, repeat=1)
        assert (out["energy"], out["count_mod_2_64"]) == _expect("config3 ising 24x24 seed 1")


def test_config4b_full_size_cube_all_leaves(bb):
    from paper_2602_05470_b200 import time_to_solve as T
    inst = I.ising_lattice_3d(5, 5, 5, 1)
    fixed = I.layer_fixed_set_3d(5, 5, 5, 8)
    tree = I.elimination_tree(inst.input_index_sets(fixed), I.min_degree_order(inst, fixed))
    out = T.solve_branched("config4b", inst, fixed, tree, repeat=1)
    assert (out["energy"], out["count_mod_2_64"]) == _expect("config4b ising 5x5x5 seed 1")


@pytest.mark.parametrize("L", [16, 20, 24])
def test_config5_shape_kings_branch_and_bound(bb, L):
    # config 5's pipeline (K5 bounds + host B&B + batched leaves) at the sizes it reaches this round
    from paper_2602_05470_b200 import time_to_solve as T
    out = T.solve_king_bb(L)
    assert (out["energy"], out["count_mod_2_64"]) == _expect(f"config5-shape king {L}x{L} p0.8 seed 1")
    assert out["leaves_contracted"] + out["nodes_pruned"] <= out["nodes_generated"]


def test_config1_config2_full_size_goldens(bb):
    for seed in (1, 2):
        e, c = bb.Handle(I.ising_lattice_2d(6, 6, seed)).contract_batch()
        assert (int(e[0]), int(c[0])) == _expect(f"config1 ising 6x6 seed {seed}")
    e, c = bb.Handle(I.kings_subgraph(12, 12, 0.8, 1)).contract_batch()
    assert (int(e[0]), int(c[0])) == _expect("config2 king 12x12 p0.8 seed 1")


# ---- BBTN proper: rho-driven non-uniform branching (bbtn_solve_branching), leaves of different fixed sets ----
@pytest.mark.parametrize("name,make,t,flags", [
    ("king10", lambda: I.kings_subgraph(10, 10, 0.8, 2), 6, 0),
    ("king12", lambda: I.kings_subgraph(12, 12, 0.8, 3), 7, 0),
    ("king9-crt", lambda: I.kings_subgraph(9, 9, 1.0, 0), 5, 1),
    ("ising6", lambda: I.ising_lattice_2d(6, 6, 4), 3, 0),
    ("cube3-crt", lambda: I.ising_lattice_3d(3, 3, 3, 2), 5, 1),
])
def test_solve_branching_matches_oracle(bb, oracle, name, make, t, flags):
    inst = make()
    ref_e, ref_c = oracle.frontier_dp(inst)
    h = bb.Handle(inst, flags=flags)
    out = h.solve_branching(t)
    assert out["rho_root"] > 0 and out["leaves"] > 1
    assert (out["energy"], out["count"]) == (ref_e, ref_c & MASK64)
    if flags:
        assert out["count_mod"] == (ref_c % 2147483647, ref_c % 2147483629)
    one = h.solve_branching(24)                    # target above the width: a single unbranched leaf
    assert one["leaves"] == 1 and (one["energy"], one["count"]) == (ref_e, ref_c & MASK64)
    h.close()


def test_solve_branching_king28_rank30_leaf(bb):
    # one rank-30 leaf (12.9 GB tensors, 0.46 TB streamed): element offsets beyond 2^30
    h = bb.Handle(I.kings_subgraph(28, 28, 0.8, 1))
    out = h.solve_branching(30)
    assert out["leaves"] == 1
    assert (out["energy"], out["count"]) == _expect("config5-shape king 28x28 p0.8 seed 1")
    out = h.solve_branching(28)                    # two leaves of different fixed sets
    assert out["leaves"] == 2
    assert (out["energy"], out["count"]) == _expect("config5-shape king 28x28 p0.8 seed 1")
    h.close()


def test_solve_branching_king32_seed2_rank31_crt(bb):
    # T_target = 2^31 as in the paper: one unbranched rank-31 leaf, count 5.3e24 > 2^64 via CRT
    g = _goldens()["config5-shape king 32x32 p0.8 seed 2"]
    h = bb.Handle(I.kings_subgraph(32, 32, 0.8, 2), flags=1)
    out = h.solve_branching(31)
    c = int(g["count"])
    assert out["leaves"] == 1 and out["energy"] == int(g["energy"]) and out["count"] == c & MASK64
    assert out["count_mod"] == (c % 2147483647, c % 2147483629)
    assert bb.crt_combine(out["count"], *out["count_mod"]) == c
    h.close()


def test_solve_branching_king32_seed1_rank32_leaves(bb):
    # T_target = 2^32: four leaves of different fixed sets, rank-32 tensors (51.5 GB each, 129 GB arena --
    # if less device memory is free the driver keeps branching, the result is the same)
    h = bb.Handle(I.kings_subgraph(32, 32, 0.8, 1))
    out = h.solve_branching(32)
    assert out["leaves"] >= 4 and out["rho_root"] == 5
    assert (out["energy"], out["count"]) == _expect("config5-shape king 32x32 p0.8 seed 1")
    h.close()


# ---- BBTN on sub-networks: local fixed sets per overflowing stretch of the tree (bbtn_solve_local) ----
@pytest.mark.parametrize("name,make,t,t2,flags,own_tree", [
    ("king10", lambda: I.kings_subgraph(10, 10, 0.8, 2), 6, 5, 0, False),
    ("king12-crt", lambda: I.kings_subgraph(12, 12, 0.8, 3), 9, 8, 1, False),
    ("king12-sweep", lambda: I.kings_subgraph(12, 12, 0.8, 4, weights="rand"), 11, 10, 0, True),
    ("king9-full-crt", lambda: I.kings_subgraph(9, 9, 1.0, 0), 9, None, 1, True),
    ("ising8", lambda: I.ising_lattice_2d(8, 8, 4), 7, None, 0, True),
    ("ising10-field-crt", lambda: I.ising_lattice_2d_half_field(10, 10, 7), 9, 8, 1, False),
    ("cube3-crt", lambda: I.ising_lattice_3d(3, 3, 3, 2), 6, 4, 1, False),
    ("cube4", lambda: I.ising_lattice_3d(4, 4, 3, 5), 13, 12, 0, True),
    ("random-mis", lambda: I.random_graph(26, 0.2, 9, "mis"), 6, 4, 1, False),
    ("king12-many-branches", lambda: I.kings_subgraph(12, 12, 0.8, 3), 8, 7, 0, False),      # 1029 and 8197 branches planned
])
def test_solve_local_matches_oracle(bb, oracle, name, make, t, t2, flags, own_tree):
    inst = make()
    ref_e, ref_c = oracle.frontier_dp(inst)
    tree = I.elimination_tree(inst.input_index_sets(), I.natural_order(inst.n_vertices)) if own_tree else None
    h = bb.Handle(inst, tree=tree, flags=flags)
    out = h.solve_local(t)
    assert out["sliced_stretches"] >= 1 and out["max_fixed"] >= 1 and out["max_rank"] <= t, out
    # every planned branch of a sliced stretch is either contracted or skipped as infeasible (run-once stretches count 1 each)
    assert out["branches_contracted"] + out["branches_infeasible"] == out["branches_planned"] - (out["stretches"] - out["sliced_stretches"])
    assert (out["energy"], out["count"]) == (ref_e, ref_c & MASK64), (name, out)
    if flags:
        assert out["count_mod"] == (ref_c % bb.BBTN_P1, ref_c % bb.BBTN_P2)
    one = h.solve_local(30)                        # threshold above the width: a single stretch that runs once
    assert one["sliced_stretches"] == 0 and one["branches_contracted"] == 0
    assert (one["energy"], one["count"]) == (ref_e, ref_c & MASK64)
    # a smaller threshold means more, smaller branches and the same result (the number of branches grows fast once the
    # threshold is far below the width: thresholds are kept within 1..3 of it)
    if t2 is not None:
        two = h.solve_local(t2)
        assert two["max_rank"] <= t2 and two["branches_planned"] > out["branches_planned"]
        # the surviving branches of a stretch run as batches (one plan, the batch axis of K1/K3), not one by one
        if two["branches_contracted"] >= 8:
            assert two["branches_in_flight"] > 1
            assert two["launch_sequences"] < two["branches_contracted"] + two["stretches"]
        assert (two["energy"], two["count"]) == (ref_e, ref_c & MASK64)
    h.close()


@pytest.mark.parametrize("kind", ["mis", "ising"])
def test_solve_local_prunes_with_region_bounds(bb, oracle, kind):
    # global pruning inside the local-branching driver: with K5 regions and an incumbent, branches whose
    # bound is strictly worse are never contracted; ties are kept, so the count stays exact (reading A14)
    if kind == "mis":
        rows = cols = 12
        inst = I.kings_subgraph(rows, cols, 0.8, 5)
        ids = _king_ids(inst, rows, cols)
    else:
        rows = cols = 9
        inst = I.ising_lattice_2d(rows, cols, 8, field_h=1)
        ids = None
    offs, verts = _grid_regions(rows, cols, 3, 3, ids)
    ref_e, ref_c = oracle.frontier_dp(inst)
    h = bb.Handle(inst, flags=bb.BBTN_COUNT_CRT)
    t = 9 if kind == "mis" else 8
    plain = h.solve_local(t)
    exact = h.solve_local(t, region_offsets=offs, region_vertices=verts, incumbent_hint=ref_e)
    loose = h.solve_local(t, region_offsets=offs, region_vertices=verts, incumbent_hint=ref_e + (3 if kind == "ising" else -3))
    for out in (plain, exact, loose):
        assert (out["energy"], out["count"]) == (ref_e, ref_c & MASK64)
        assert out["count_mod"] == (ref_c % bb.BBTN_P1, ref_c % bb.BBTN_P2)
        assert out["branches_contracted"] + out["branches_infeasible"] + out["branches_pruned"] == \
            out["branches_planned"] - (out["stretches"] - out["sliced_stretches"])
    assert plain["branches_pruned"] == 0 and exact["branches_pruned"] >= loose["branches_pruned"]
    assert exact["branches_contracted"] <= plain["branches_contracted"]
    h.close()


@pytest.mark.parametrize("L,seed,t", [(28, 1, 29), (32, 1, 31), (32, 2, 30), (36, 1, 32), (36, 2, 32), (36, 3, 32)])
def test_solve_local_kings_large(bb, L, seed, t):
    # King's subgraphs at filling 0.8 beyond the reach of one dense contraction at the threshold: goldens by the
    # oracle's sparse frontier DP (tests/golden/config_goldens.json)
    g = _goldens()[f"config5-shape king {L}x{L} p0.8 seed {seed}"]
    c = int(g["count"])
    k = I.kings_subgraph(L, L, 0.8, seed)
    h = bb.Handle(k, flags=bb.BBTN_COUNT_CRT)
    if seed != 1:
        h.add_sweep_order(I.column_major_order(k))      # a hint for the tree search: sweeps along the columns as well
    out = h.solve_local(t)
    assert out["energy"] == int(g["energy"]) and out["count"] == c & MASK64, out
    assert out["count_mod"] == (c % bb.BBTN_P1, c % bb.BBTN_P2)
    assert bb.crt_combine(out["count"], *out["count_mod"]) == c
    h.close()


@pytest.mark.parametrize("seed", [1, 2])
def test_config5_kings_40x40_exact_size_and_count(bb, seed):
    # BASELINE configs[4]: MIS on the King's subgraph 40x40, filling 0.8, unit weights: exact size and count (1.1e32 for
    # seed 1, so all three residues are needed) by local branching, with K5 region bounds on every branch
    g = _goldens()[f"config5 king 40x40 p0.8 seed {seed}"]
    c = int(g["count"])
    k = I.kings_subgraph(40, 40, 0.8, seed)
    offs, verts = _grid_regions(40, 40, 4, 4, _king_ids(k, 40, 40))
    h = bb.Handle(k, flags=bb.BBTN_COUNT_CRT)
    h.add_sweep_order(I.column_major_order(k))
    out = h.solve_local(32, region_offsets=offs, region_vertices=verts, incumbent_hint=int(g["energy"]))
    assert out["energy"] == int(g["energy"]) and out["count"] == c & MASK64, out
    assert bb.crt_combine(out["count"], *out["count_mod"]) == c
    h.close()


# ---- ground-state SEARCH mode: plain max-plus, no count plane (BBTN_SEARCH_ONLY) ----
@pytest.mark.parametrize("case", range(5))
def test_search_mode_energies_match_oracle(bb, oracle, case):
    # PAPER.md:55 ("the tropical number inf for optimization problems"), :81-91: the optimum alone.  Every leaf energy must
    # equal the counting oracle's energy (max-plus without counts is its energy half); counts read 0
    if case == 0:
        inst = I.ising_lattice_2d(7, 8, 3, field_h=1)
    elif case == 1:
        inst = I.kings_subgraph(8, 8, 0.8, 4, weights="rand")          # weighted MIS
    elif case == 2:
        inst = I.ising_lattice_3d(3, 3, 4, 5)
    elif case == 3:
        inst = I.random_graph(22, 0.2, 7, "mis")
    else:
        inst = I.kings_subgraph(4, 4, 1.0, 1)                          # infeasible leaves
    n = inst.n_vertices
    fixed = np.array([0, 1, 5], np.int32) if case == 4 else I.random_order(n, 70 + case)[:4]
    assign = I.all_assignments(len(fixed))
    for tree, extra in ((None, 0), (I.elimination_tree(inst.input_index_sets(), I.natural_order(n)), 0),
                        (None, bb.BBTN_FORCE_TILED | bb.BBTN_NO_FUSED)):       # permute + max-plus GEMM wherever an index is summed
        h = bb.Handle(inst, tree=tree, flags=bb.BBTN_SEARCH_ONLY | extra)
        energy, count = h.contract_batch(fixed, assign)
        assert (count == 0).all()
        for b in range(len(assign)):
            we, _ = oracle.frontier_dp(inst, None, fixed, assign[b])
            assert int(energy[b]) == (NEG_INF if we is None else we), (case, b)
        e1, _ = h.contract_batch()
        assert int(e1[0]) == oracle.frontier_dp(inst)[0]
        h.close()


def test_search_mode_drivers_and_large_kings(bb, oracle):
    # the solve drivers in search mode: host B&B with K5 pruning, rho-driven branching, local branching
    k = I.kings_subgraph(12, 12, 0.8, 5, weights="rand")
    want = oracle.frontier_dp(k)[0]
    ids = _king_ids(k, 12, 12)
    offs, verts = _grid_regions(12, 12, 3, 3, ids)
    branch = np.array([ids[r][6] for r in range(12) if ids[r][6] >= 0], np.int32)
    h = bb.Handle(k, flags=bb.BBTN_SEARCH_ONLY)
    assert h.solve_bb(branch, 3, offs, verts, max_batch=64)["energy"] == want
    assert h.solve_branching(7)["energy"] == want
    out = h.solve_local(9, region_offsets=offs, region_vertices=verts, incumbent_hint=want)
    assert out["energy"] == want and out["count"] == 0 and out["sliced_stretches"] >= 1
    with pytest.raises(bb.BbtnError):
        bb.Handle(k, flags=bb.BBTN_SEARCH_ONLY | bb.BBTN_COUNT_CRT)
    h.close()
    # MIS size of the 36x36 and 40x40 King's subgraphs (goldens by the oracle's sparse DP): 4 B per element
    for L, seed, name in ((36, 1, "config5-shape king 36x36 p0.8 seed 1"), (40, 1, "config5 king 40x40 p0.8 seed 1"),
                          (40, 3, "config5 king 40x40 p0.8 seed 3")):
        k = I.kings_subgraph(L, L, 0.8, seed)
        h = bb.Handle(k, flags=bb.BBTN_SEARCH_ONLY)
        if seed != 1:
            h.add_sweep_order(I.column_major_order(k))
        out = h.solve_local(32)
        assert out["energy"] == int(_goldens()[name]["energy"]) and out["count"] == 0, out
        h.close()


@pytest.mark.parametrize("B,M,N,K,seed,frac", [
    (1, 64, 64, 64, 61, 0.0),
    (3, 256, 256, 256, 62, 0.0),
    (2, 131, 197, 100, 63, 0.2),          # ragged in every dimension, zero elements
    (5, 1, 1, 1, 64, 0.0),
    (1, 129, 65, 513, 65, 0.05),
    (4, 17, 201, 3, 66, 0.5),             # odd leading dimension: the scalar load/store paths
    (1, 1, 300, 1000, 67, 0.0),
    (2, 333, 1, 129, 68, 0.3),
    (7, 48, 64, 33, 69, 0.2),             # M, N <= 64: the 64x64 tile, ragged, batched
    (3, 64, 37, 70, 70, 0.0),
    (1, 300, 129, 17, 71, 0.9),           # mostly zero elements: whole rows / columns of -inf
])
def test_maxplus_gemm_matches_oracle(bb, oracle, B, M, N, K, seed, frac):
    # K3 of the search mode alone: max-plus on the energy plane = the energy half of the counting oracle's GEMM
    import torch
    Ae, Ac, Be, Bc = I.gemm_operands(B, M, N, K, seed, neg_inf_frac=frac)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    prev = bb.set_debug_checks(True)
    try:
        want_e, _ = _oracle_gemm(oracle, Ae, Ac, Be, Bc)
        for ebits in (7, 32):                                          # packed 16-bit halves / 32-bit
            assert (bb.maxplus_gemm_batched(dev(Ae), dev(Be), energy_bits=ebits).cpu().numpy() == want_e).all(), ebits
        # the whole range of the packed form (-2047..2047) and the zero element
        spread = lambda e, sft: np.where(e <= -(1 << 29), e, ((e.astype(np.int64) * 31 + sft) % 4095 - 2047)).astype(np.int32)
        A2, B2 = spread(Ae, 7), spread(Be, 1900)
        want2, _ = _oracle_gemm(oracle, A2, Ac, B2, Bc)
        for ebits in (11, 12, 32):
            assert (bb.maxplus_gemm_batched(dev(A2), dev(B2), energy_bits=ebits).cpu().numpy() == want2).all(), ebits
        if A2.size > 100 and frac < 0.5:
            with pytest.raises(bb.BbtnError):                          # |e| up to 2047 is not below 2^10
                bb.maxplus_gemm_batched(dev(A2), dev(B2), energy_bits=10)
        # energies up to +-2^27 (sums within the finite range): the 32-bit form
        big = lambda e: np.where(e <= -(1 << 29), e, e.astype(np.int64) * (1 << 15)).astype(np.int32)
        A3, B3 = big(A2), big(B2)
        want3, _ = _oracle_gemm(oracle, A3, Ac, B3, Bc)
        assert (bb.maxplus_gemm_batched(dev(A3), dev(B3), energy_bits=27).cpu().numpy() == want3).all()
    finally:
        bb.set_debug_checks(prev)
    # a shared operand (stride 0) holding non-canonical zero elements (anything below -2^29 reads as zero)
    if B > 1:
        Bz = Be[0].copy(); Bz[Bz <= -(1 << 29)] = -(1 << 29) - 5
        wants, _ = _oracle_gemm(oracle, Ae, Ac, np.broadcast_to(Be[0], Be.shape).copy(), np.broadcast_to(Bc[0], Bc.shape).copy())
        for ebits in (7, 32):
            assert (bb.maxplus_gemm_batched(dev(Ae), dev(Bz), energy_bits=ebits).cpu().numpy() == wants).all(), ebits


@pytest.mark.parametrize("case", ["ising12", "king12", "ising12-sliced", "king12-sliced"])
def test_search_mode_block_tree_runs_permute_and_maxplus_gemm(bb, oracle, case):
    # the divide-and-conquer trees of test_block_tree_runs_tiled_gemm_and_trace_kernels in search mode: the joins are
    # energy-only K2 + the max-plus K3 (automatic mode); every leaf energy equals the counting oracle's
    L = 12
    if case.startswith("ising"):
        inst = I.ising_lattice_2d(L, L, 3)
        ids = None
    else:
        inst = I.kings_subgraph(L, L, 1.0, 6, weights="rand")
        ids = _king_ids(inst, L, L)
    fixed, assign = None, None
    if case.endswith("sliced"):
        v = lambda r, c: r * L + c if ids is None else int(ids[r][c])
        fixed = np.array([v(2, 2), v(2, L - 3), v(L - 3, 3)], np.int32)
        assign = I.all_assignments(3)
    parts = I.lattice_block_parts(L, L, [L // 2], [L // 2], ids, exclude=() if fixed is None else fixed)
    tree = I.grouped_elimination_tree(inst.input_index_sets(() if fixed is None else fixed), parts)
    for flags in (bb.BBTN_SEARCH_ONLY, bb.BBTN_SEARCH_ONLY | bb.BBTN_FORCE_TILED | bb.BBTN_NO_GRAPH):
        h = bb.Handle(inst, tree=tree, flags=flags)
        info = h.plan_query(fixed, 1 if assign is None else len(assign))
        assert info["n_gemm_tiled"] > 0 and info["n_permute"] > 0, info
        energy, count = h.contract_batch(fixed, assign)
        assert (count == 0).all()
        for b in range(len(energy)):
            we, _ = oracle.contract_tree(inst, tree[0], tree[1], fixed, None if assign is None else assign[b])
            assert int(energy[b]) == we, (case, flags, b)
        h.close()


@pytest.mark.parametrize("L", [16, 20, 24])
def test_paper_e1_spin_glass_with_half_field(bb, L):
    # +-J with external field 0.5, in integers (J -> 2J, h -> 1, half units; reading A6): one unbranched
    # leaf through bbtn_solve_branching, and all 2^8 leaves of a slit through bbtn_contract_batch
    inst = I.ising_lattice_2d_half_field(L, L, 1)
    want = _expect(f"paper-E1 ising {L}x{L} seed 1 h=0.5 (2J, h=1, half units)")
    h = bb.Handle(inst)
    out = h.solve_branching(31)
    assert out["leaves"] == 1 and (out["energy"], out["count"]) == want
    fixed = I.slit_fixed_set_2d(L, L, 8)
    e, c = h.contract_batch(fixed, I.all_assignments(8))
    assert bb.oplus_combine("ising", e, c)[:2] == want
    h.close()
