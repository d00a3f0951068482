"""Thin ctypes binding over the C ABI of include/bbtn.h (libbbtn.so).

Argument marshalling only: every step of the path runs in the CUDA kernels.
PyTorch appears here for device memory and streams (device-pointer entry
points); host-pointer entry points take numpy arrays.  There is no CPU
fallback: a missing library raises at load time, a missing device makes every
compute call fail with BBTN_ECUDA.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libbbtn.so")
_lib = None

BBTN_OK, BBTN_EINVAL, BBTN_ENOMEM, BBTN_ECUDA, BBTN_ESHAPE, BBTN_ERANGE = range(6)
BBTN_NEG_INF = -(1 << 30)
BBTN_COUNT_CRT, BBTN_IO_DEVICE, BBTN_NO_GRAPH = 0x1, 0x2, 0x4
BBTN_FORCE_STREAMING, BBTN_FORCE_TILED, BBTN_SEARCH_ONLY, BBTN_NO_FUSED = 0x10, 0x20, 0x40, 0x80
BBTN_P1, BBTN_P2 = 2147483647, 2147483629

EXPORTS = ["bbtn_build", "bbtn_contract_batch", "bbtn_plan_query", "bbtn_region_bound", "bbtn_region_bound_static", "bbtn_solve_bb", "bbtn_solve_branching", "bbtn_branching_leaves", "bbtn_solve_local", "bbtn_local_plan_query", "bbtn_add_sweep_order",
           "bbtn_tropical_gemm_batched", "bbtn_tropical_gemm_batched_host", "bbtn_maxplus_gemm_batched", "bbtn_oplus_combine",
           "bbtn_permute_batched", "bbtn_int32_microbench", "bbtn_crt_combine", "bbtn_set_debug_checks",
           "bbtn_destroy", "bbtn_last_error", "bbtn_version"]


class BbtnError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"bbtn status {status}: {msg}")
        self.status = status


class _Desc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_vertices", C.c_int32), ("n_edges", C.c_int32),
                ("edge_u", C.c_void_p), ("edge_v", C.c_void_p), ("edge_w", C.c_void_p), ("vertex_w", C.c_void_p),
                ("n_steps", C.c_int32), ("tree_l", C.c_void_p), ("tree_r", C.c_void_p),
                ("max_elements_per_leaf", C.c_int64), ("flags", C.c_uint32)]


class _PlanInfo(C.Structure):
    _fields_ = [("n_nodes", C.c_int32), ("n_variant_nodes", C.c_int32), ("max_rank", C.c_int32),
                ("n_gemm_tiled", C.c_int32), ("n_absorb", C.c_int32), ("n_permute", C.c_int32), ("n_trace", C.c_int32),
                ("rho", C.c_int64), ("fma_variant", C.c_double), ("fma_invariant", C.c_double),
                ("bytes_per_call", C.c_double), ("workspace_bytes", C.c_int64),
                ("n_kernel_launches", C.c_int32), ("reserved", C.c_int32)]


def load():
    """Load libbbtn.so (built in-tree by paper_2602_05470_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2602_05470_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.bbtn_build.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]
    lib.bbtn_contract_batch.argtypes = [vp, vp, i32, vp, i64, vp, vp, vp, vp]
    lib.bbtn_plan_query.argtypes = [vp, vp, i32, i64, C.POINTER(_PlanInfo)]
    lib.bbtn_region_bound.argtypes = [vp, vp, vp, i32, vp, i32, vp, i64, vp, vp]
    lib.bbtn_region_bound_static.argtypes = [vp, vp, vp, i32, vp, i32, vp, i64, vp, vp]
    lib.bbtn_solve_bb.argtypes = [vp, vp, i32, i32, vp, vp, i32, i64, i32, i32, vp, vp, vp, vp, vp]
    lib.bbtn_solve_branching.argtypes = [vp, i32, i64, i64, vp, vp, vp, vp, vp, vp]
    lib.bbtn_branching_leaves.argtypes = [vp, i32, i64, i64, i64, i64, vp, vp, vp, vp, vp]
    lib.bbtn_solve_local.argtypes = [vp, i32, i64, vp, vp, i32, i32, vp, vp, vp, vp, vp, vp]
    lib.bbtn_local_plan_query.argtypes = [vp, i32, i64, vp, vp]
    lib.bbtn_add_sweep_order.argtypes = [vp, vp]
    lib.bbtn_tropical_gemm_batched.argtypes = [i64, i32, i32, i32, vp, vp, vp, vp, vp, vp, i64, i64, i64, i32, i32, vp]
    lib.bbtn_maxplus_gemm_batched.argtypes = [i64, i32, i32, i32, vp, vp, vp, i64, i64, i64, i32, vp]
    lib.bbtn_tropical_gemm_batched_host.argtypes = [i64, i32, i32, i32, vp, vp, vp, vp, vp, vp, i64, i64, i64, i32, i32, vp]
    lib.bbtn_oplus_combine.argtypes = [i32, i64, vp, vp, vp, vp, vp, vp]
    lib.bbtn_permute_batched.argtypes = [i32, vp, i64, vp, vp, vp, vp, vp]
    lib.bbtn_int32_microbench.argtypes = [i32, i32, C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
    lib.bbtn_crt_combine.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, vp]
    lib.bbtn_set_debug_checks.argtypes = [i32]
    lib.bbtn_destroy.argtypes = [vp]
    lib.bbtn_destroy.restype = None
    lib.bbtn_last_error.argtypes = [vp]
    lib.bbtn_last_error.restype = C.c_char_p
    lib.bbtn_version.restype = C.c_char_p
    _lib = lib
    return lib


def _np(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


def _ptr(a):
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()          # torch tensor


def _check(rc, h=None):
    if rc != BBTN_OK:
        raise BbtnError(rc, load().bbtn_last_error(h).decode())


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else None
    return stream


class Handle:
    """bbtn_build / bbtn_destroy + the batched calls.  `inst` is an instances.Instance."""

    def __init__(self, inst, tree=None, max_elements_per_leaf: int = 0, flags: int = 0):
        lib = load()
        self._keep = [_np(inst.edge_u, np.int32), _np(inst.edge_v, np.int32), _np(inst.edge_w, np.int32),
                      _np(inst.vertex_w, np.int32)]
        tl = tr = None
        if tree is not None:
            tl, tr = _np(tree[0], np.int32), _np(tree[1], np.int32)
        d = _Desc(0 if inst.kind == "ising" else 1, inst.n_vertices, inst.n_edges, _ptr(self._keep[0]),
                  _ptr(self._keep[1]), _ptr(self._keep[2]), _ptr(self._keep[3]),
                  0 if tl is None else len(tl), _ptr(tl), _ptr(tr), max_elements_per_leaf, flags)
        self._h = C.c_void_p()
        self.flags = flags
        self.kind = inst.kind
        _check(lib.bbtn_build(C.byref(d), C.byref(self._h)))

    def close(self):
        if self._h:
            load().bbtn_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- bbtn_contract_batch, host pointers
    def contract_batch(self, fixed=None, assign=None, B: int | None = None, stream=None):
        lib = load()
        fx = np.zeros(0, np.int32) if fixed is None else _np(fixed, np.int32)
        asg = None if assign is None else _np(assign, np.uint8)
        if B is None:
            B = 1 if asg is None else int(asg.shape[0])
        if asg is not None and len(fx):
            assert asg.shape == (B, len(fx))
        energy = np.empty(B, np.int32); count = np.empty(B, np.uint64)
        cm = np.empty((B, 2), np.uint32) if self.flags & BBTN_COUNT_CRT else None
        _check(lib.bbtn_contract_batch(self._h, _ptr(fx), len(fx), _ptr(asg), B, _ptr(energy), _ptr(count), _ptr(cm),
                                       _stream(stream)), self._h)
        return (energy, count, cm) if cm is not None else (energy, count)

    # -- bbtn_contract_batch, device pointers (handle built with BBTN_IO_DEVICE); torch tensors
    def contract_batch_device(self, fixed, assign_t, energy_t, count_t, count_mod_t=None, stream=None):
        lib = load()
        fx = np.zeros(0, np.int32) if fixed is None else _np(fixed, np.int32)
        B = int(energy_t.shape[0])
        _check(lib.bbtn_contract_batch(self._h, _ptr(fx), len(fx), _ptr(assign_t), B, _ptr(energy_t), _ptr(count_t),
                                       _ptr(count_mod_t), _stream(stream)), self._h)

    def plan_query(self, fixed=None, B: int = 1) -> dict:
        fx = np.zeros(0, np.int32) if fixed is None else _np(fixed, np.int32)
        info = _PlanInfo()
        _check(load().bbtn_plan_query(self._h, _ptr(fx), len(fx), B, C.byref(info)), self._h)
        return {k: getattr(info, k) for k, _ in _PlanInfo._fields_}

    def region_bound(self, region_offsets, region_vertices, fixed=None, assign=None, B: int | None = None, stream=None):
        ro, rv = _np(region_offsets, np.int32), _np(region_vertices, np.int32)
        fx = np.zeros(0, np.int32) if fixed is None else _np(fixed, np.int32)
        asg = None if assign is None else _np(assign, np.uint8)
        if B is None:
            B = 1 if asg is None else int(asg.shape[0])
        bound = np.empty(B, np.int32)
        _check(load().bbtn_region_bound(self._h, _ptr(ro), _ptr(rv), len(ro) - 1, _ptr(fx), len(fx), _ptr(asg), B,
                                        _ptr(bound), _stream(stream)), self._h)
        return bound

    # -- bbtn_region_bound, device pointers (handle built with BBTN_IO_DEVICE); torch tensors
    def region_bound_device(self, region_offsets, region_vertices, fixed, assign_t, bound_t, stream=None):
        ro, rv = _np(region_offsets, np.int32), _np(region_vertices, np.int32)
        fx = np.zeros(0, np.int32) if fixed is None else _np(fixed, np.int32)
        _check(load().bbtn_region_bound(self._h, _ptr(ro), _ptr(rv), len(ro) - 1, _ptr(fx), len(fx), _ptr(assign_t),
                                        int(bound_t.shape[0]), _ptr(bound_t), _stream(stream)), self._h)

    # -- bbtn_region_bound_static: no device allocation; device tensors whatever the handle's flags; B = 0 is the set-up call
    def region_bound_static(self, region_offsets, region_vertices, fixed, assign_t, bound_t, B: int | None = None, stream=None):
        ro, rv = _np(region_offsets, np.int32), _np(region_vertices, np.int32)
        fx = np.zeros(0, np.int32) if fixed is None else _np(fixed, np.int32)
        if B is None:
            B = int(bound_t.shape[0])
        _check(load().bbtn_region_bound_static(self._h, _ptr(ro), _ptr(rv), len(ro) - 1, _ptr(fx), len(fx), _ptr(assign_t),
                                               B, _ptr(bound_t), _stream(stream)), self._h)

    def solve_bb(self, branch_vertices, chunk, region_offsets, region_vertices, max_batch=1024,
                 incumbent_hint=BBTN_NEG_INF, use_pruning=True, stream=None):
        bv = _np(branch_vertices, np.int32)
        ro, rv = _np(region_offsets, np.int32), _np(region_vertices, np.int32)
        e = C.c_int32(); c = C.c_uint64(); cm = (C.c_uint32 * 2)(); stats = (C.c_int64 * 4)()
        crt = bool(self.flags & BBTN_COUNT_CRT)
        _check(load().bbtn_solve_bb(self._h, _ptr(bv), len(bv), chunk, _ptr(ro), _ptr(rv), len(ro) - 1, max_batch,
                                    incumbent_hint, 1 if use_pruning else 0, C.addressof(e), C.addressof(c),
                                    C.addressof(cm) if crt else None, C.addressof(stats), _stream(stream)), self._h)
        out = {"energy": e.value, "count": c.value, "generated": stats[0], "pruned": stats[1],
               "contracted": stats[2], "calls": stats[3]}
        if crt:
            out["count_mod"] = (cm[0], cm[1])
        return out


    def solve_branching(self, log2_target: int, mem_budget_bytes: int = 0, max_leaves: int = 0, stream=None):
        """bbtn_solve_branching: rho-driven non-uniform branching (Eq. 4), leaves contracted on the device."""
        e = C.c_int32(); c = C.c_uint64(); cm = (C.c_uint32 * 2)(); stats = (C.c_int64 * 4)(); work = (C.c_double * 2)()
        crt = bool(self.flags & BBTN_COUNT_CRT)
        _check(load().bbtn_solve_branching(self._h, log2_target, mem_budget_bytes, max_leaves, C.addressof(e),
                                           C.addressof(c), C.addressof(cm) if crt else None, C.addressof(stats),
                                           C.addressof(work), _stream(stream)), self._h)
        out = {"energy": e.value, "count": c.value, "branch_nodes": stats[0], "leaves": stats[1],
               "max_fixed": stats[2], "rho_root": stats[3], "fma": work[0], "bytes": work[1]}
        if crt:
            out["count_mod"] = (cm[0], cm[1])
        return out

    _LOCAL_STATS = ("stretches", "sliced_stretches", "branches_planned", "branches_contracted", "branches_infeasible",
                    "branches_pruned", "max_fixed", "max_rank", "arena_bytes", "kernel_launches", "branches_in_flight",
                    "launch_sequences")

    def solve_local(self, log2_target: int, mem_budget_bytes: int = 0, region_offsets=None, region_vertices=None,
                    incumbent_hint=BBTN_NEG_INF, stream=None):
        """bbtn_solve_local: BBTN on sub-networks (local fixed sets per overflowing stretch of the tree)."""
        e = C.c_int32(); c = C.c_uint64(); cm = (C.c_uint32 * 2)(); stats = (C.c_int64 * 12)(); work = (C.c_double * 4)()
        crt = bool(self.flags & BBTN_COUNT_CRT)
        ro = None if region_offsets is None else _np(region_offsets, np.int32)
        rv = None if region_vertices is None else _np(region_vertices, np.int32)
        _check(load().bbtn_solve_local(self._h, log2_target, mem_budget_bytes, _ptr(ro), _ptr(rv), 0 if ro is None else len(ro) - 1,
                                       incumbent_hint, C.addressof(e), C.addressof(c), C.addressof(cm) if crt else None,
                                       C.addressof(stats), C.addressof(work), _stream(stream)), self._h)
        out = {"energy": e.value, "count": c.value, "fma": work[0], "bytes": work[1], "fma_contracted": work[2],
               "bytes_contracted": work[3]}
        out.update({k: stats[i] for i, k in enumerate(self._LOCAL_STATS)})
        if crt:
            out["count_mod"] = (cm[0], cm[1])
        return out

    def add_sweep_order(self, order):
        """bbtn_add_sweep_order: another base order (a permutation of the vertices) for the library's tree search."""
        o = _np(order, np.int32)
        _check(load().bbtn_add_sweep_order(self._h, _ptr(o)), self._h)

    def local_plan_query(self, log2_target: int, mem_budget_bytes: int = 0) -> dict:
        """bbtn_local_plan_query (host only)."""
        stats = (C.c_int64 * 12)(); work = (C.c_double * 4)()
        _check(load().bbtn_local_plan_query(self._h, log2_target, mem_budget_bytes, C.addressof(stats), C.addressof(work)), self._h)
        out = {"fma": work[0], "bytes": work[1]}
        out.update({k: stats[i] for i, k in enumerate(self._LOCAL_STATS)})
        return out

    def branching_leaves(self, log2_target: int, mem_budget_bytes: int = 0, max_leaves: int = 0, store: bool = True,
                         cap_entries: int = 1 << 24):
        """bbtn_branching_leaves (host only): the leaves [(fixed vertices, values)] and the stats."""
        stats = (C.c_int64 * 4)(); work = (C.c_double * 2)()
        if not store:
            _check(load().bbtn_branching_leaves(self._h, log2_target, mem_budget_bytes, max_leaves, 0, 0, None, None,
                                                None, C.addressof(stats), C.addressof(work)), self._h)
            leaves = None
        else:
            cap_leaves = max(max_leaves, 1 << 16)
            off = np.zeros(cap_leaves + 1, np.int64); lv = np.zeros(cap_entries, np.int32); lx = np.zeros(cap_entries, np.uint8)
            _check(load().bbtn_branching_leaves(self._h, log2_target, mem_budget_bytes, max_leaves, cap_leaves, cap_entries,
                                                _ptr(off), _ptr(lv), _ptr(lx), C.addressof(stats), C.addressof(work)), self._h)
            leaves = [(lv[off[i]:off[i + 1]].copy(), lx[off[i]:off[i + 1]].copy()) for i in range(stats[1])]
        return leaves, {"branch_nodes": stats[0], "leaves": stats[1], "max_fixed": stats[2], "rho_root": stats[3],
                        "fma": work[0], "bytes": work[1]}


def tropical_gemm_batched(Ae, Ac, Be, Bc, Ce=None, Cc=None, count_bits: int = 64, energy_bits: int = 32, stream=None):
    """bbtn_tropical_gemm_batched on torch CUDA tensors: A [B][M][K] (or [M][K] shared), B [B][K][N]
    (or [K][N] shared); energies int32, counts int64 storage (bit pattern of uint64)."""
    import torch
    a3, b3 = Ae.dim() == 3, Be.dim() == 3
    batch = Ae.shape[0] if a3 else (Be.shape[0] if b3 else 1)
    M, K = Ae.shape[-2:]
    N = Be.shape[-1]
    assert Be.shape[-2] == K
    if Ce is None:
        Ce = torch.empty((batch, M, N), dtype=torch.int32, device=Ae.device)
        Cc = torch.empty((batch, M, N), dtype=torch.int64, device=Ae.device)
    _check(load().bbtn_tropical_gemm_batched(batch, M, N, K, _ptr(Ae), _ptr(Ac), _ptr(Be), _ptr(Bc), _ptr(Ce), _ptr(Cc),
                                             M * K if a3 else 0, K * N if b3 else 0, M * N, count_bits, energy_bits, _stream(stream)))
    return Ce, Cc


def maxplus_gemm_batched(A, B, C=None, energy_bits: int = 32, stream=None):
    """bbtn_maxplus_gemm_batched on torch CUDA int32 tensors: A [B][M][K] (or [M][K] shared), B [B][K][N] (or [K][N])."""
    import torch
    a3, b3 = A.dim() == 3, B.dim() == 3
    batch = A.shape[0] if a3 else (B.shape[0] if b3 else 1)
    M, K = A.shape[-2:]
    N = B.shape[-1]
    assert B.shape[-2] == K
    if C is None:
        C = torch.empty((batch, M, N), dtype=torch.int32, device=A.device)
    _check(load().bbtn_maxplus_gemm_batched(batch, M, N, K, _ptr(A), _ptr(B), _ptr(C), M * K if a3 else 0, K * N if b3 else 0,
                                            M * N, energy_bits, _stream(stream)))
    return C


def tropical_gemm_batched_host(Ae, Ac, Be, Bc, Ce=None, Cc=None, count_bits: int = 64, energy_bits: int = 32, stream=None):
    """bbtn_tropical_gemm_batched_host: same layouts on HOST arrays (numpy, or pinned CPU torch tensors with
    int64 storage for the counts); copies in, runs K3, copies C back."""
    shp = lambda a: tuple(a.shape)
    a3, b3 = len(shp(Ae)) == 3, len(shp(Be)) == 3
    batch = shp(Ae)[0] if a3 else (shp(Be)[0] if b3 else 1)
    M, K = shp(Ae)[-2:]
    N = shp(Be)[-1]
    assert shp(Be)[-2] == K
    if Ce is None:
        Ce = np.empty((batch, M, N), np.int32); Cc = np.empty((batch, M, N), np.uint64)
    _check(load().bbtn_tropical_gemm_batched_host(batch, M, N, K, _ptr(Ae), _ptr(Ac), _ptr(Be), _ptr(Bc), _ptr(Ce), _ptr(Cc),
                                                  M * K if a3 else 0, K * N if b3 else 0, M * N, count_bits, energy_bits, _stream(stream)))
    return Ce, Cc


def oplus_combine(kind, energy, count, count_mod=None):
    """bbtn_oplus_combine: (+) over leaf results in reported units (Eq. 3's outer sum).  Host only."""
    e = _np(energy, np.int32); c = _np(count, np.uint64)
    cm = None if count_mod is None else _np(count_mod, np.uint32)
    oe = C.c_int32(); oc = C.c_uint64(); om = (C.c_uint32 * 2)()
    k = {"ising": 0, "mis": 1, 0: 0, 1: 1}[kind]
    _check(load().bbtn_oplus_combine(k, len(e), _ptr(e), _ptr(c), _ptr(cm), C.addressof(oe), C.addressof(oc),
                                     C.addressof(om) if cm is not None else None))
    return (oe.value, oc.value) if cm is None else (oe.value, oc.value, (om[0], om[1]))


def permute_batched(perm, src_e, src_c, dst_e=None, dst_c=None, stream=None):
    """bbtn_permute_batched on torch CUDA tensors [B][2^r]."""
    import torch
    p = _np(perm, np.int32)
    batch = src_e.shape[0]
    assert src_e.shape[1] == 1 << len(p)
    if dst_e is None:
        dst_e = torch.empty_like(src_e); dst_c = torch.empty_like(src_c)
    _check(load().bbtn_permute_batched(len(p), _ptr(p), batch, _ptr(src_e), _ptr(src_c), _ptr(dst_e), _ptr(dst_c),
                                       _stream(stream)))
    return dst_e, dst_c


def int32_microbench(which: int, iters: int = 2000, stream=None):
    """Returns (milliseconds, operations)."""
    ms = C.c_double(); ops = C.c_double()
    _check(load().bbtn_int32_microbench(which, iters, C.byref(ms), C.byref(ops), _stream(stream)))
    return ms.value, ops.value


def crt_combine(c64: int, r1: int, r2: int) -> int:
    """bbtn_crt_combine: (count mod 2^64, mod P1, mod P2) -> count mod 2^64*P1*P2 (reading A9), as a Python int
    assembled from the two 64-bit limbs the library returns."""
    out = (C.c_uint64 * 2)()
    _check(load().bbtn_crt_combine(int(c64), int(r1), int(r2), C.addressof(out)))
    return int(out[0]) | (int(out[1]) << 64)


def set_debug_checks(on: bool) -> bool:
    """bbtn_set_debug_checks: verify the raw GEMM's count_bits / energy-range promises on the device."""
    return bool(load().bbtn_set_debug_checks(1 if on else 0))
