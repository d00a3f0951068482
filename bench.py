#!/usr/bin/env python
"""bench.py -- measurement of the BBTN hot path on B200 (contract of the driver).

    python bench.py --gpus N --steps K --warmup W [--impl reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Workload = BASELINE.json configs[3], the configuration the metric ("counting-tropical GEMM Gop/s & %
of int32 CUDA-core peak") is quoted on.  ONE STEP is one pass of the whole hot path over one batch:
  (a) raw batched counting-tropical GEMM (K3 tiled): M=N=K=1024, batch 64 per GPU, energies uniform
      in [-64,64], counts uniform in {1..4} (so the caller promises count_bits = 3 and energy_bits = 7,
      which selects the packed 16x2 form of K3);
      followed by K2 on its result: the 2^26-element C planes are bit-permuted (seeded random permutation
      of the 26 index bits) into the order a following contraction would want;
  (b) the 5x5x5 open +-J cube, 2^f leaves (f = 8 spins of the central layer, all assignments) per
      GPU: K5 region bounds for every leaf, then K1 construct -> K2 permute / K3 GEMM (tiled and
      streaming forms, chosen per tree node by the planner) -> K4 finalize.
Units: 1 tropical FMA = one (batch, m, n, k) term ((.) then (+)); Gop/s = 2 x GFMA/s.
`value` counts the planner's algorithmic FMAs (leaf-invariant nodes once), inputs resident in HBM;
`e2e` is the same step through the host-pointer C-ABI calls (H2D of operands/assignments and D2H of
results inside the timed region).  Weak scaling: every rank runs its own seeded batch; no collective
on the data path (results are 12 bytes per leaf).  Inputs are larger than L2 (no flush needed).

After the timed steps the same run also reports (untimed by the step clock, each with its own CUDA-event or
wall-clock timing, N = 1 only): `gemm_sweep` -- the corners of the config-4a sweep in every count/energy mode;
`time_to_solve` -- exact (E0, count) of configs 1, 2, 3, 4b and of King's subgraphs 36x36 and 40x40 (configs[4]),
each asserted against tests/golden/config_goldens.json inside the run; `cpu_baseline` on 1 core and on all cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2602_05470_b200 import instances as I  # noqa: E402  (seeded inputs only; no arithmetic of the method)

GEMM_N, GEMM_BATCH = 1024, 64
CUBE_L, CUBE_F = 5, 8
METRIC = "counting-tropical GEMM Gop/s (2 x tropical FMA/s) over one pass of the hot path"
# int32 lane-instructions a tropical FMA needs on this ISA:
# fused add-max, tie test = add + compare, multiply-accumulate of the counts (1 IMAD.WIDE for <=32-bit
# operand counts, 3 IMADs for full 64x64->64).
INT_OPS_PER_FMA = {32: 4, 64: 6}
# executed warp instructions per lane-FMA in the inner loop of gemm_pack16_kernel, counted in the SASS of the in-tree
# object (profiles/r2_k3_pack16_sass.md): per 128 FMAs 64 VIADDMNMX.S16x2 + 64 adds + 64 HSETP2 + 128 IMAD + 28 LDS.128 + 16 others
PACK16_INSTR_PER_FMA = 364.0 / 128.0
SWEEP = [(64, 1024), (256, 256), (1024, 64), (4096, 2)]                # (n, batch) corners of config 4a
SWEEP_MODES = [("3:7", "packed 16x2 energies, 32-bit accumulators", 32),
               ("13:7", "packed 16x2 energies, carry form (31-bit running sum + carry register), 64-bit totals", 32),
               ("32:7", "packed 16x2 energies, 32-bit operands, 64-bit accumulators", 32), ("3:32", "32-bit accumulators", 32),
               ("14:32", "chunk-local 32-bit tie sums, 64-bit accumulators", 32),
               ("32:32", "32-bit operands, 64-bit accumulators", 32), ("64:32", "full 64x64 count product", 64)]


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d.get("hbm_gbs", 6650.0), "measured", d.get("sm_max_mhz", 1965.0)
    return 6650.0, "fallback", 1965.0


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for _, r in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def cube_problem(seed: int):
    inst = I.ising_lattice_3d(CUBE_L, CUBE_L, CUBE_L, seed)
    fixed = I.layer_fixed_set_3d(CUBE_L, CUBE_L, CUBE_L, CUBE_F)
    assign = I.all_assignments(CUBE_F)
    # K5 regions: the 2x2x2-ish blocks of the cube (disjoint, <= 12 vertices each)
    offs, verts = [0], []
    L = CUBE_L
    for z0 in range(0, L, 2):
        for y0 in range(0, L, 2):
            for x0 in range(0, L, 3):
                verts += [(z * L + y) * L + x for z in range(z0, min(z0 + 2, L)) for y in range(y0, min(y0 + 2, L))
                          for x in range(x0, min(x0 + 3, L))]
                offs.append(len(verts))
    return inst, fixed, assign, np.array(offs, np.int32), np.array(verts, np.int32)


# ----------------------------------------------------------------------------------------------
# reference arm: the oracle, as it stands, on the host cores, on a bounded sample of the same step
# ----------------------------------------------------------------------------------------------
def oracle_sample(seed: int, rows: int = 32, leaves: int = 4, threads: int = 0):
    """One bounded sample of the step through oracle/: `rows` rows of one GEMM batch entry (OpenMP over
    rows) and `leaves` leaves of the cube (naive loop-nest contraction, one thread per leaf).
    Returns (tropical FMAs done, seconds, threads used, description)."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    oracle.build()
    n = GEMM_N
    Ae, Ac, Be, Bc = I.gemm_operands(1, n, n, n, seed)
    Ae, Ac = Ae[:, :rows].astype(np.int64), Ac[:, :rows]
    Be64 = Be.astype(np.int64)
    z = lambda a: np.zeros(a.shape, np.uint8)
    inst, fixed, assign, _, _ = cube_problem(seed)
    tree = _cube_tree(inst, fixed)
    cores = threads if threads > 0 else (os.cpu_count() or 1)      # threads = 1: OMP_NUM_THREADS=1 is set by the caller
    t0 = time.perf_counter()
    oracle.gemm(Ae, z(Ae), Ac, Be64, z(Be64), Bc)
    with ThreadPoolExecutor(max_workers=min(leaves, cores)) as ex:
        list(ex.map(lambda b: oracle.contract_tree(inst, tree[0], tree[1], fixed, assign[b]), range(leaves)))
    dt = time.perf_counter() - t0
    fma = float(rows) * n * n + leaves * I.tree_fma(inst.input_index_sets(fixed), tree)
    return fma, dt, cores, (f"oracle/: {rows} rows of one {n}^3 GEMM entry (OpenMP) + {leaves} of {1 << CUBE_F} cube leaves "
                            f"(naive loop-nest tree contraction, one thread each)")


def _cube_tree(inst, fixed):
    """Contraction tree of the cube used by BOTH arms: bucket elimination along a min-degree order
    (instances.py: pure graph structure)."""
    return I.elimination_tree(inst.input_index_sets(fixed), I.min_degree_order(inst, fixed))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    vals = []
    for s in range(args.warmup + args.steps):
        fma, dt, cores, desc = oracle_sample(args.seed + s, rows=args.ref_rows, leaves=args.ref_leaves)
        if s >= args.warmup:
            vals.append((fma, dt))
    tot_f = sum(f for f, _ in vals); tot_t = sum(t for _, t in vals)
    v = 2.0 * tot_f / tot_t / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "Gop/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32 energy + uint64 count (oracle: int64 + 256-bit)",
            "data": "synthetic", "config": _config(args),
            "cpu_baseline": {"value": v, "unit": "Gop/s", "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": "Gop/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def _config(args):
    return {"workload": (f"BASELINE configs[3]: raw batched counting-tropical GEMM M=N=K={GEMM_N} batch {GEMM_BATCH} "
                         f"(energies U[-64,64], counts U{{1..4}}) + K2 bit-permutation of its 2^26-element result + {CUBE_L}x{CUBE_L}x{CUBE_L} open +-J cube, "
                         f"f={CUBE_F} fixed spins of the central layer, all {1 << CUBE_F} leaves, per GPU"),
            "gemm": {"M": GEMM_N, "N": GEMM_N, "K": GEMM_N, "batch_per_gpu": GEMM_BATCH, "count_bits": 3, "energy_bits": 7},
            "cube": {"L": CUBE_L, "n_fixed": CUBE_F, "leaves_per_gpu": 1 << CUBE_F},
            "l2_policy": "inputs larger than L2 (2.4 GB of GEMM planes, multi-GB contraction arena); no flush",
            "seed": args.seed}



# ----------------------------------------------------------------------------------------------
# extras reported in the same JSON line (rank 0, N = 1): sweep corners, time-to-solve, oracle on 1 / all cores
# ----------------------------------------------------------------------------------------------
def _goldens():
    with open(os.path.join(ROOT, "tests", "golden", "config_goldens.json")) as f:
        return json.load(f)["cases"]


def gemm_sweep_block(bb, torch, stream, int_peak, viaddmnmx_peak, repeat=3):
    """Corners of the config-4a sweep (n, batch) in every count/energy mode: GFMA/s and the fraction of the int32 roof
    (4 algorithmic int32 lane-instructions per FMA; 6 for the full 64x64 count product).  Then the search mode's K3
    (max-plus on the energy planes, bbtn_maxplus_gemm_batched) on the same operands: its one instruction per FMA
    (per two FMAs in the packed form) is VIADDMNMX, so its roof is the measured VIADDMNMX issue rate."""
    out = []
    ev = lambda: torch.cuda.Event(enable_timing=True)
    for n, B in SWEEP:
        gen = min(B, 4)
        Ae, Ac, Be, Bc = I.gemm_operands(gen, n, n, n, seed=1000 * n + B)
        rep = lambda x: torch.from_numpy(x.view(np.int64) if x.dtype == np.uint64 else x).cuda().repeat((B + gen - 1) // gen, 1, 1)[:B].contiguous()
        dAe, dAc, dBe, dBc = rep(Ae), rep(Ac), rep(Be), rep(Bc)
        dCe = torch.empty((B, n, n), dtype=torch.int32, device="cuda"); dCc = torch.empty((B, n, n), dtype=torch.int64, device="cuda")
        ref = None
        for mode, what, acc_bits in SWEEP_MODES:
            bits, ebits = (int(x) for x in mode.split(":"))
            ts = []
            with torch.cuda.stream(stream):
                for it in range(repeat + 1):
                    a, b = ev(), ev()
                    a.record(stream)
                    bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, dCe, dCc, count_bits=bits, energy_bits=ebits, stream=stream.cuda_stream)
                    b.record(stream); b.synchronize()
                    if it:
                        ts.append(a.elapsed_time(b))
            chk = (int(dCe.sum().item()), int(dCc.sum().item()))      # every mode must give the same integers
            ref = ref or chk
            assert chk == ref, f"GEMM modes disagree at n={n}: {mode}"
            ms = float(np.median(ts))
            gfma = float(B) * n ** 3 / ms / 1e6
            out.append({"n": n, "batch": B, "mode": mode, "what": what, "ms": ms, "gfma_per_s": gfma,
                        "frac_of_int32_peak": INT_OPS_PER_FMA[acc_bits] * gfma / int_peak})
        dCm = torch.empty_like(dCe)
        for ebits, what, fma_per_instr in ((7, "search mode: max-plus, packed 16-bit energies", 2), (32, "search mode: max-plus, 32-bit energies", 1)):
            ts = []
            with torch.cuda.stream(stream):
                for it in range(repeat + 1):
                    a, b = ev(), ev()
                    a.record(stream)
                    bb.maxplus_gemm_batched(dAe, dBe, dCm, energy_bits=ebits, stream=stream.cuda_stream)
                    b.record(stream); b.synchronize()
                    if it:
                        ts.append(a.elapsed_time(b))
            assert bool((dCm == dCe).all().item()), f"max-plus GEMM disagrees with the energies of the counting GEMM at n={n}"
            ms = float(np.median(ts))
            gfma = float(B) * n ** 3 / ms / 1e6
            out.append({"n": n, "batch": B, "mode": f"0:{ebits}", "what": what, "ms": ms, "gfma_per_s": gfma,
                        "frac_of_viaddmnmx_peak": gfma / fma_per_instr / viaddmnmx_peak})
        del dAe, dAc, dBe, dBc, dCe, dCc, dCm
    return out


def time_to_solve_block(bb, skip_king40=False):
    """Second half of the metric: time to the exact (E0, count), each result asserted against the oracle's goldens."""
    from paper_2602_05470_b200 import time_to_solve as T
    g = _goldens()
    mask = (1 << 64) - 1
    out = []

    def check(name, rec, energy, c64, full=None):
        want = g[name]
        assert energy == int(want["energy"]) and c64 == int(want["count"]) & mask, (name, energy, c64, want)
        if full is not None:
            assert int(full) == int(want["count"]), (name, full, want["count"])
        rec["golden"] = name; rec["exact"] = True
        out.append(rec)

    r = T.solve_unbranched("config1 ising 6x6 seed 1", I.ising_lattice_2d(6, 6, 1))
    check("config1 ising 6x6 seed 1", {"config": 1, "ms": r["ms_median"], "width": r["width"], "launches": r["kernel_launches"]}, r["energy"], r["count_mod_2_64"])
    r = T.solve_unbranched("config2 king 12x12 p0.8 seed 1", I.kings_subgraph(12, 12, 0.8, 1))
    check("config2 king 12x12 p0.8 seed 1", {"config": 2, "ms": r["ms_median"], "width": r["width"], "launches": r["kernel_launches"]}, r["energy"], r["count_mod_2_64"])
    inst = I.ising_lattice_2d(24, 24, 1)
    for f in (8, 10, 12):
        fixed = I.slit_fixed_set_2d(24, 24, f)
        tree = I.elimination_tree(inst.input_index_sets(fixed), I.slit_angular_order_2d(24, 24, f))
        r = T.solve_branched("config3", inst, fixed, tree, repeat=3)
        check("config3 ising 24x24 seed 1", {"config": 3, "n_fixed": f, "leaves": r["leaves"], "ms": r["ms_median"], "width": r["width"],
                                             "algorithmic_gb_per_s": r["algorithmic_gb_per_s"]}, r["energy"], r["count_mod_2_64"])
    inst = I.ising_lattice_3d(5, 5, 5, 1)
    fixed = I.layer_fixed_set_3d(5, 5, 5, 8)
    tree = I.elimination_tree(inst.input_index_sets(fixed), I.min_degree_order(inst, fixed))
    r = T.solve_branched("config4b", inst, fixed, tree, repeat=3)
    check("config4b ising 5x5x5 seed 1", {"config": "4b", "n_fixed": 8, "leaves": r["leaves"], "ms": r["ms_median"], "width": r["width"],
                                          "algorithmic_gb_per_s": r["algorithmic_gb_per_s"]}, r["energy"], r["count_mod_2_64"])
    for L, name in ((36, "config5-shape king 36x36 p0.8 seed 1"), (40, "config5 king 40x40 p0.8 seed 1")):
        if L == 40 and skip_king40:
            continue
        r = T.solve_king_local(L, 1, 32, crt=True, hint=int(g[name]["energy"]))
        check(name, {"config": 5, "king": L, "seconds": r["seconds"], "plan_seconds": r["plan_only_seconds"],
                     "mode": "bbtn_solve_local, T_target 2^32, three count residues in two passes (mod 2^64; p1 and p2 packed), K5 bounds vs the golden optimum as incumbent",
                     **{k: r[k] for k in ("stretches", "sliced_stretches", "branches_planned", "branches_contracted", "branches_infeasible",
                                          "branches_pruned", "max_fixed", "max_rank", "arena_bytes", "kernel_launches")},
                     "algorithmic_gb_per_s": r["algorithmic_gb_per_s"], "count": r["count"]}, r["energy"], r["count_mod_2_64"], r["count"])
    return out


def cpu_baseline_both(args):
    """The oracle on the host: all cores in-process, one core in a child process (OMP_NUM_THREADS=1)."""
    fma, dt, cores, desc = oracle_sample(args.seed, rows=args.ref_rows, leaves=args.ref_leaves)
    res = {"value": 2.0 * fma / dt / 1e9, "unit": "Gop/s", "cores": cores, "kind": "oracle", "sample": desc, "seconds": dt}
    try:
        env = dict(os.environ, OMP_NUM_THREADS="1")
        rows1, leaves1 = max(8, args.ref_rows // 8), max(1, args.ref_leaves // 8)
        o = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-sample", f"{args.seed}:{rows1}:{leaves1}"],
                           env=env, capture_output=True, text=True, timeout=600)
        one = json.loads(o.stdout.strip().splitlines()[-1])
        res["one_core"] = {"value": one["gops"], "unit": "Gop/s", "cores": 1, "seconds": one["seconds"], "sample": one["sample"]}
    except Exception as e:                      # the single-core figure is a nicety; never lose the line over it
        res["one_core"] = {"error": repr(e)}
    return res


def _traffic_from_profile():
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed ncu capture."""
    p = os.path.join(ROOT, "profiles", "r2_k3_dram_traffic.csv")
    try:
        rows = [l.strip().split(",") for l in open(p) if l.strip() and not l.startswith("#")]
        hdr, val = rows[0], rows[1]
        d = dict(zip(hdr, val))
        return float(d["dram_bytes_read"]) + float(d["dram_bytes_write"]), f"profiles/r2_k3_dram_traffic.csv ({d.get('kernel', '?')}, ncu --set full)"
    except Exception:
        return None, "no committed capture found"

# ----------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2602_05470_b200 import binding as bb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    bb.load()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm_peak, peak_kind, sm_max = _peaks()
    seed = args.seed + 1000 * rank
    stream = torch.cuda.Stream()
    sp = stream.cuda_stream

    # ---- inputs (a): GEMM planes, resident in HBM
    n, gb = GEMM_N, GEMM_BATCH
    Ae, Ac, Be, Bc = I.gemm_operands(gb, n, n, n, seed)
    pin = lambda a: torch.from_numpy(a.view(np.int64) if a.dtype == np.uint64 else a).pin_memory()
    hAe, hAc, hBe, hBc = pin(Ae), pin(Ac), pin(Be), pin(Bc)
    dAe, dAc, dBe, dBc = (t.cuda(non_blocking=True) for t in (hAe, hAc, hBe, hBc))
    dCe = torch.empty((gb, n, n), dtype=torch.int32, device="cuda")
    dCc = torch.empty((gb, n, n), dtype=torch.int64, device="cuda")
    hCe = torch.empty((gb, n, n), dtype=torch.int32).pin_memory()
    hCc = torch.empty((gb, n, n), dtype=torch.int64).pin_memory()
    gemm_fma = float(gb) * n * n * n
    perm_rank = int(np.log2(gb * n * n))
    perm = I.random_bit_permutation(perm_rank, seed)
    dPe = torch.empty((1, gb * n * n), dtype=torch.int32, device="cuda")
    dPc = torch.empty((1, gb * n * n), dtype=torch.int64, device="cuda")
    perm_bytes = 24.0 * gb * n * n

    # ---- inputs (b): cube
    inst, fixed, assign, roffs, rverts = cube_problem(seed)
    tree = _cube_tree(inst, fixed)
    B = len(assign)
    h_dev = bb.Handle(inst, tree=tree, max_elements_per_leaf=1 << 26, flags=bb.BBTN_IO_DEVICE)
    h_host = bb.Handle(inst, tree=tree, max_elements_per_leaf=1 << 26)
    info = h_dev.plan_query(fixed, B)
    cube_fma = info["fma_variant"] * B + info["fma_invariant"]
    d_assign = torch.from_numpy(assign).cuda()
    d_energy = torch.empty(B, dtype=torch.int32, device="cuda")
    d_count = torch.empty(B, dtype=torch.int64, device="cuda")
    d_bound = torch.empty(B, dtype=torch.int32, device="cuda")
    step_fma = gemm_fma + cube_fma
    launches_per_step = 1 + 1 + 2 + info["n_kernel_launches"]

    ev = lambda: torch.cuda.Event(enable_timing=True)
    gemm_ev, perm_ev, cube_ev = [], [], []

    def step_device(record=False):
        with torch.cuda.stream(stream):
            h_dev.region_bound_device(roffs, rverts, fixed, d_assign, d_bound, stream=sp)
            if record:
                c0, c1, a, b, q = ev(), ev(), ev(), ev(), ev()
                c0.record(stream)
            h_dev.contract_batch_device(fixed, d_assign, d_energy, d_count, stream=sp)
            if record:
                c1.record(stream)
                a.record(stream)
            bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, dCe, dCc, count_bits=3, energy_bits=7, stream=sp)
            if record:
                b.record(stream)
            bb.permute_batched(perm, dCe.view(1, -1), dCc.view(1, -1), dPe, dPc, stream=sp)
            if record:
                q.record(stream)
                gemm_ev.append((a, b)); perm_ev.append((b, q)); cube_ev.append((c0, c1))

    def step_host():
        bound = h_host.region_bound(roffs, rverts, fixed, assign, stream=sp)
        e, c = h_host.contract_batch(fixed, assign, stream=sp)
        bb.tropical_gemm_batched_host(hAe, hAc, hBe, hBc, hCe, hCc, count_bits=3, energy_bits=7, stream=sp)
        return bound, e, c

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    for _ in range(args.warmup):
        step_device()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    t_wall0 = time.time()
    e0, e1 = ev(), ev()
    e0.record(stream)
    for _ in range(args.steps):
        step_device(record=True)
    e1.record(stream)
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    ms = e0.elapsed_time(e1)
    gemm_ms = float(np.mean([a.elapsed_time(b) for a, b in gemm_ev]))
    perm_ms = float(np.mean([a.elapsed_time(b) for a, b in perm_ev]))
    cube_ms = float(np.mean([a.elapsed_time(b) for a, b in cube_ev]))
    energy_dev = d_energy.cpu().numpy().copy(); count_dev = d_count.cpu().numpy().copy()

    # ---- the timed outputs are checked, not only produced: the packed GEMM result must equal, element for element, what the
    #      general 32-bit / 64-bit-count form gives on the same operands, and pi^-1 after pi must return the GEMM planes
    with torch.cuda.stream(stream):
        rCe = torch.empty_like(dCe); rCc = torch.empty_like(dCc)
        bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, rCe, rCc, count_bits=64, energy_bits=32, stream=sp)
        qe, qc = bb.permute_batched(np.argsort(perm).astype(np.int32), dPe, dPc, stream=sp)
    torch.cuda.synchronize()
    gemm_ok = bool(torch.equal(rCe, dCe) and torch.equal(rCc, dCc))
    perm_ok = bool(torch.equal(qe.view(-1), dCe.view(-1)) and torch.equal(qc.view(-1), dCc.view(-1)))
    assert gemm_ok and perm_ok, "timed K3 / K2 outputs failed their cross-checks"
    del rCe, rCc, qe, qc

    # ---- end-to-end timing through the host-pointer calls
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    for _ in range(min(args.warmup, 2)):
        step_host()
    barrier()
    a, b = ev(), ev()
    a.record(stream)
    for _ in range(e2e_steps):
        bound, e_h, c_h = step_host()
    b.record(stream)
    barrier()
    ms_e2e = a.elapsed_time(b)
    assert (e_h == energy_dev).all() and (c_h.view(np.int64) == count_dev).all(), "host and device paths disagree"
    h2d = Ae.nbytes + Ac.nbytes + Be.nbytes + Bc.nbytes + 2 * assign.nbytes
    d2h = hCe.numel() * 4 + hCc.numel() * 8 + B * (4 + 8 + 4)

    if world > 1:
        t = torch.tensor([ms, ms_e2e, gemm_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, ms_e2e, gemm_ms = (float(x) for x in t.cpu())
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    value = 2.0 * step_fma * world * args.steps / (ms * 1e-3) / 1e9
    e2e_value = 2.0 * step_fma * world * e2e_steps / (ms_e2e * 1e-3) / 1e9

    # ---- ALU roofline of the dominant kernel (K3 tiled GEMM), against the committed microbenchmark
    mb = {}
    for which, name in ((0, "iadd3"), (1, "imnmx"), (2, "viaddmnmx"), (3, "imad"), (4, "iadd3+imad"), (7, "iadd+imad_2op"),
                        (8, "2iadd+imad_2op"), (9, "k3mix_2warps"), (10, "k3mix_4warps")):
        t_ms, ops = bb.int32_microbench(which, args.microbench_iters if which < 9 else max(args.microbench_iters // 16, 50))
        mb[name] = ops / (t_ms * 1e-3) / 1e9          # G lane-ops/s (which <= 8) or GFMA/s (K3 instruction mix)
    # building blocks of the packed / 64-bit forms: clocks per warp instruction (or per round) on one SM sub-partition
    blocks = {}
    for which, name in ((11, "VIADDMNMX.S16x2"), (12, "HSETP2+SEL"), (13, "ISETP+SEL"), (14, "IMAD.WIDE (64-bit accumulate)"),
                        (15, "packed pair = 2 FMAs: VIADDMNMX.S16x2 + add + HSETP2 + 2 @p IMAD")):
        t_ms, rounds = bb.int32_microbench(which, max(args.microbench_iters // 4, 100))
        blocks[name] = 1.0 / (rounds / 32 / (148 * 4) / (t_ms * 1e-3) / (sm_max * 1e6))
    int_peak = max(mb[k] for k in ("iadd3+imad", "iadd+imad_2op", "2iadd+imad_2op", "iadd3", "imnmx", "imad"))
    alu_peak = max(mb["iadd3"], mb["imnmx"], mb["viaddmnmx"])
    gemm_gfma = gemm_fma / (gemm_ms * 1e-3) / 1e9
    achieved = INT_OPS_PER_FMA[32] * gemm_gfma
    traffic, traffic_src = _traffic_from_profile()
    issue_peak = 148 * 4 * 32 * (clocks["sm_mhz"] or sm_max) * 1e6 / 1e9 if clocks else None   # G lane-instructions/s the schedulers can issue
    roofline = {"bound": "alu", "kernel": "gemm_pack16_kernel (K3, packed 16x2 form)", "achieved": achieved, "peak": int_peak, "unit": "Gop/s",
                "frac": achieved / int_peak,
                "traffic": traffic, "traffic_source": traffic_src,
                "traffic_unit": "bytes per launch (algorithmic operand+result bytes: %.3e)" % (3.0 * gb * n * n * 12),
                "note": (f"op = int32 lane-operation; achieved = {INT_OPS_PER_FMA[32]} ALGORITHMIC int32 operations per tropical FMA "
                         "(add-max, tie add, tie compare, multiply-add of the counts) x GFMA/s of the K3 launch; peak = committed "
                         "microbenchmark (bbtn_int32_microbench), best of IADD3 / IMNMX / IMAD / mixed ALU+FMA-pipe issue of SCALAR int32 "
                         "instructions, same run.  The packed form executes 2.5 instructions per FMA (VIADDMNMX.S16x2 and HSETP2 handle two "
                         "outputs each), so `frac` can exceed what scalar int32 code could reach; `executed_frac_of_issue_peak` = "
                         "instructions actually issued (SASS count per FMA x GFMA/s) over the schedulers' issue limit is the utilisation figure"),
                "executed_instr_per_fma": PACK16_INSTR_PER_FMA,
                "executed_frac_of_issue_peak": (PACK16_INSTR_PER_FMA * gemm_gfma / issue_peak) if issue_peak else None,
                "gemm_gfma_per_s": gemm_gfma, "gemm_gop_per_s": 2 * gemm_gfma, "gemm_ms_per_launch": gemm_ms,
                "frac_of_scalar_opmix_ceiling": gemm_gfma / max(mb["k3mix_2warps"], mb["k3mix_4warps"]),
                "frac_of_alu_pipe_peak_2ops": 2 * gemm_gfma / alu_peak,
                "microbench_Gops": mb, "microbench_clk_per_warp_round_per_smsp": blocks, "share_of_step": gemm_ms * args.steps / ms,
                "hbm_peak_gbs": hbm_peak, "hbm_peak_kind": peak_kind}
    # the HBM-bound kernels of the same step (rank 0's timings), against the measured copy bandwidth
    roofline_hbm = [
        {"kernel": "permute_vec_kernel (K2)", "bound": "hbm", "achieved": perm_bytes / perm_ms / 1e6, "peak": hbm_peak,
         "unit": "GB/s", "frac": perm_bytes / perm_ms / 1e6 / hbm_peak, "ms_per_launch": perm_ms,
         "algorithmic_bytes": perm_bytes, "what": f"2^{perm_rank} elements x 24 B (12 read + 12 written), seeded random bit permutation"},
        {"kernel": "absorb_vec/absorb_stage kernels + shared-memory prologue + K1/K2/K4 (S1-S4 of the cube, one CUDA-graph replay)", "bound": "hbm",
         "achieved": info["bytes_per_call"] / cube_ms / 1e6, "peak": hbm_peak, "unit": "GB/s",
         "frac": info["bytes_per_call"] / cube_ms / 1e6 / hbm_peak, "ms_per_call": cube_ms,
         "algorithmic_bytes": info["bytes_per_call"], "what": "planner byte total: 12 B per element read or written by every tree node"}]

    # ---- the oracle beside it (bounded sample, rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_both(args)
    sweep = tts = None
    if world == 1 and not args.no_extras:
        sweep = gemm_sweep_block(bb, torch, stream, int_peak, mb["viaddmnmx"])
        h_dev.close(); h_host.close()
        del dAe, dAc, dBe, dBc, dCe, dCc, dPe, dPc
        torch.cuda.empty_cache()
        tts = time_to_solve_block(bb, skip_king40=args.skip_king40)

    line = {"metric": METRIC, "value": value, "unit": "Gop/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int32 energy + uint64 count (K3 computes the energies as packed s16x2 under the caller's |e| < 2^7 promise)",
            "data": "synthetic", "config": _config(args),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "Gop/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "note": "host-pointer calls: region_bound + contract_batch + tropical_gemm_batched_host (K2 has no host-pointer form and is left out)",
                    "ms_per_step": ms_e2e / e2e_steps, "steps": e2e_steps},
            "gpu_launches": int(launches_per_step * args.steps),
            "roofline": roofline, "roofline_hbm_kernels": roofline_hbm, "cpu_baseline": cpu,
            "gemm_sweep": sweep, "time_to_solve": tts,
            "plan": {k: info[k] for k in ("n_nodes", "n_variant_nodes", "max_rank", "n_gemm_tiled", "n_absorb", "n_permute",
                                          "n_trace", "n_kernel_launches", "workspace_bytes")},
            "fma_per_step": {"gemm": gemm_fma, "cube": cube_fma},
            "result_check": {"timed_gemm_equals_general_form": gemm_ok, "timed_permute_inverts": perm_ok, "cube_E0": int(energy_dev.min()),
                             "cube_count_mod_2_64": int(sum(int(x) for x in count_dev.view(np.uint64)[energy_dev == energy_dev.min()]) & ((1 << 64) - 1))}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--ref-rows", type=int, default=128)
    ap.add_argument("--ref-leaves", type=int, default=16)
    ap.add_argument("--microbench-iters", type=int, default=4000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the gemm_sweep and time_to_solve blocks")
    ap.add_argument("--skip-king40", action="store_true", help="leave the ~1.5 min King 40x40 solve out of time_to_solve")
    ap.add_argument("--oracle-sample", default=None, help=argparse.SUPPRESS)     # child of cpu_baseline_both: seed:rows:leaves
    args = ap.parse_args()
    if args.oracle_sample:
        seed, rows, leaves = (int(x) for x in args.oracle_sample.split(":"))
        fma, dt, cores, desc = oracle_sample(seed, rows=rows, leaves=leaves, threads=1)
        print(json.dumps({"gops": 2.0 * fma / dt / 1e9, "seconds": dt, "sample": desc}))
        return 0
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3          # timing rule: W >= 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
