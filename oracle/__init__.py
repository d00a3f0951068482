"""CPU oracle for the BBTN hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes wrapper over oracle/bbtn_oracle.c (plain C, compiled with gcc).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` leg may import this package.  It imports nothing from
paper_2602_05470_b200 and shares no code with the CUDA path.

Every function takes the problem in the C-ABI's own terms (edge lists, integer
couplings/weights, SSA tree, fixed set + one assignment) and returns Python
ints, so counts are exact big integers (256-bit in C).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bbtn_oracle.c")
_SO = os.path.join(_HERE, "libbbtn_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (OpenMP for the DP and GEMM loops)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    with _lock:
        if _lib is None:
            _lib = C.CDLL(build())
    return _lib


def _i32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


def _p(a, t=C.c_void_p):
    return None if a is None else a.ctypes.data_as(t)


def _count(c4) -> int:
    return int(c4[0]) | (int(c4[1]) << 64) | (int(c4[2]) << 128) | (int(c4[3]) << 192)


def _kind(kind) -> int:
    return {"ising": 0, "mis": 1, 0: 0, 1: 1}[kind]


def _common(inst):
    eu, ev = _i32(inst.edge_u), _i32(inst.edge_v)
    ew, vw = _i32(inst.edge_w), _i32(inst.vertex_w)
    return eu, ev, ew, vw


def _fixed(fixed, assign):
    fx = np.zeros(0, np.int32) if fixed is None else _i32(fixed)
    asg = np.zeros(0, np.uint8) if assign is None else np.ascontiguousarray(assign, dtype=np.uint8)
    assert asg.shape[0] == fx.shape[0]
    return fx, asg


def exhaustive(inst, fixed=None, assign=None):
    """Definition (Eq. 1 / Eq. 2; MIS :55).  Returns (energy, count);
    energy is None for an infeasible MIS assignment (zero element)."""
    lib = _load()
    eu, ev, ew, vw = _common(inst)
    fx, asg = _fixed(fixed, assign)
    e = C.c_int64(); f = C.c_int32(); c4 = (C.c_uint64 * 4)()
    rc = lib.oracle_exhaustive(_kind(inst.kind), inst.n_vertices, inst.n_edges, _p(eu), _p(ev), _p(ew), _p(vw),
                               len(fx), _p(fx), _p(asg), C.byref(e), C.byref(f), c4)
    if rc:
        raise RuntimeError(f"oracle_exhaustive rc={rc}")
    return (e.value if f.value else None), _count(c4)


def contract_tree(inst, tree_l, tree_r, fixed=None, assign=None, return_rank=False):
    """Eq. 2 evaluated pairwise along the SSA tree, sliced per Eq. 3."""
    lib = _load()
    eu, ev, ew, vw = _common(inst)
    fx, asg = _fixed(fixed, assign)
    tl, tr = _i32(tree_l), _i32(tree_r)
    e = C.c_int64(); f = C.c_int32(); c4 = (C.c_uint64 * 4)(); mr = C.c_int32()
    rc = lib.oracle_contract_tree(_kind(inst.kind), inst.n_vertices, inst.n_edges, _p(eu), _p(ev), _p(ew), _p(vw),
                                  len(tl), _p(tl), _p(tr), len(fx), _p(fx), _p(asg),
                                  C.byref(e), C.byref(f), c4, C.byref(mr))
    if rc:
        raise RuntimeError(f"oracle_contract_tree rc={rc}")
    out = ((e.value if f.value else None), _count(c4))
    return out + (mr.value,) if return_rank else out


def frontier_dp(inst, order=None, fixed=None, assign=None, return_width=False):
    """Independent exact method: transfer/frontier DP over `order` (all vertices)."""
    lib = _load()
    eu, ev, ew, vw = _common(inst)
    fx, asg = _fixed(fixed, assign)
    od = np.arange(inst.n_vertices, dtype=np.int32) if order is None else _i32(order)
    assert len(od) == inst.n_vertices
    e = C.c_int64(); f = C.c_int32(); c4 = (C.c_uint64 * 4)(); mf = C.c_int32()
    rc = lib.oracle_frontier_dp(_kind(inst.kind), inst.n_vertices, inst.n_edges, _p(eu), _p(ev), _p(ew), _p(vw),
                                _p(od), len(fx), _p(fx), _p(asg), C.byref(e), C.byref(f), c4, C.byref(mf))
    if rc:
        raise RuntimeError(f"oracle_frontier_dp rc={rc}")
    out = ((e.value if f.value else None), _count(c4))
    return out + (mf.value,) if return_width else out


def frontier_dp_mis_sparse(inst, order=None, fixed=None, assign=None, return_stats=False):
    """oracle-3 for MIS with only the independent frontier states stored;
    reaches King's subgraphs whose dense frontier table would not fit.  Returns (size, count)."""
    assert _kind(inst.kind) == 1
    lib = _load()
    eu, ev, _, vw = _common(inst)
    fx, asg = _fixed(fixed, assign)
    od = np.arange(inst.n_vertices, dtype=np.int32) if order is None else _i32(order)
    assert len(od) == inst.n_vertices
    e = C.c_int64(); f = C.c_int32(); c4 = (C.c_uint64 * 4)(); mf = C.c_int32(); ms = C.c_int64()
    rc = lib.oracle_frontier_dp_mis_sparse(inst.n_vertices, inst.n_edges, _p(eu), _p(ev), _p(vw), _p(od),
                                           len(fx), _p(fx), _p(asg), C.byref(e), C.byref(f), c4,
                                           C.byref(mf), C.byref(ms))
    if rc:
        raise RuntimeError(f"oracle_frontier_dp_mis_sparse rc={rc}")
    out = ((e.value if f.value else None), _count(c4))
    return out + (mf.value, ms.value) if return_stats else out


def gemm(Ae, Az, Ac, Be, Bz, Bc, full_counts=False):
    """C[b,m,n] = (+)_k A[b,m,k] (.) B[b,k,n].  A* are [B][M][K], B* are [B][K][N].
    Energies int64, zero flags uint8, counts uint64.  Returns (Ce, Cz, Cc mod 2^64[, Cc4])."""
    lib = _load()
    Ae = np.ascontiguousarray(Ae, np.int64); Be = np.ascontiguousarray(Be, np.int64)
    Az = np.ascontiguousarray(Az, np.uint8); Bz = np.ascontiguousarray(Bz, np.uint8)
    Ac = np.ascontiguousarray(Ac, np.uint64); Bc = np.ascontiguousarray(Bc, np.uint64)
    Bn, M, K = Ae.shape
    _, K2, N = Be.shape
    assert K2 == K and Be.shape[0] == Bn
    Ce = np.zeros((Bn, M, N), np.int64); Cz = np.zeros((Bn, M, N), np.uint8); Cc = np.zeros((Bn, M, N), np.uint64)
    Cc4 = np.zeros((Bn, M, N, 4), np.uint64) if full_counts else None
    lib.oracle_gemm.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_int] + [C.c_void_p] * 10
    rc = lib.oracle_gemm(Bn, M, N, K, _p(Ae), _p(Az), _p(Ac), _p(Be), _p(Bz), _p(Bc), _p(Ce), _p(Cz), _p(Cc), _p(Cc4))
    if rc:
        raise RuntimeError(f"oracle_gemm rc={rc}")
    return (Ce, Cz, Cc, Cc4) if full_counts else (Ce, Cz, Cc)


def permute(perm, src_e, src_c):
    """dst[pi(i)] = src[i]; bit j of pi(i) = bit perm[j] of i.  src_* are [B][2^r]."""
    lib = _load()
    perm = _i32(perm)
    src_e = np.ascontiguousarray(src_e, np.int32); src_c = np.ascontiguousarray(src_c, np.uint64)
    Bn = src_e.shape[0]
    dst_e = np.empty_like(src_e); dst_c = np.empty_like(src_c)
    lib.oracle_permute.argtypes = [C.c_int, C.c_void_p, C.c_int64] + [C.c_void_p] * 4
    lib.oracle_permute(len(perm), _p(perm), Bn, _p(src_e), _p(src_c), _p(dst_e), _p(dst_c))
    return dst_e, dst_c


def region_bound(inst, region_offsets, region_vertices, fixed=None, assign=None):
    """Pruning bound, reading A15, in max-plus units
    (Ising: an upper bound on -H; MIS: on the set weight).  None if infeasible."""
    lib = _load()
    eu, ev, ew, vw = _common(inst)
    fx, asg = _fixed(fixed, assign)
    ro, rv = _i32(region_offsets), _i32(region_vertices)
    b = C.c_int64(); inf = C.c_int32()
    rc = lib.oracle_region_bound(_kind(inst.kind), inst.n_vertices, inst.n_edges, _p(eu), _p(ev), _p(ew), _p(vw),
                                 len(ro) - 1, _p(ro), _p(rv), len(fx), _p(fx), _p(asg), C.byref(b), C.byref(inf))
    if rc:
        raise RuntimeError(f"oracle_region_bound rc={rc}")
    return None if inf.value else b.value


def rho(log2_sizes, log2_target) -> int:
    """Eq. 4."""
    lib = _load()
    a = _i32(log2_sizes)
    lib.oracle_rho.restype = C.c_int64
    return int(lib.oracle_rho(len(a), _p(a), int(log2_target)))


# (+) over leaf results in REPORTED units (Eq. 3's outer sum):
# oplus_min for Ising energies (min H), oplus_max for MIS weights.
def oplus_min(results):
    best, cnt = None, 0
    for e, c in results:
        if e is None:
            continue
        if best is None or e < best:
            best, cnt = e, c
        elif e == best:
            cnt += c
    return best, cnt


def oplus_max(results):
    best, cnt = None, 0
    for e, c in results:
        if e is None:
            continue
        if best is None or e > best:
            best, cnt = e, c
        elif e == best:
            cnt += c
    return best, cnt
