"""World-size-2 checks on CPU (gloo) of the parts of the path that involve more than one process:
the leaf sharding + final (+) of DESIGN.md section 8 (Eq. 3: leaves are independent), and the
launch contract of `bench.py --impl reference` under torchrun (rank 0 prints one line, the others exit 0)."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_path):
    # leaves of one branching are dealt round-robin to the ranks; every rank (+)-combines its own leaf results with
    # bbtn_oplus_combine, then the per-rank partials are all-gathered and combined the same way (12 bytes per rank)
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import oracle
    from paper_2602_05470_b200 import binding as bb, instances as I
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    bb.load()
    inst = I.kings_subgraph(8, 8, 0.8, 1)
    h = bb.Handle(inst)
    leaves, st = h.branching_leaves(5)
    mine = leaves[rank::world]
    res = [oracle.frontier_dp(inst, fixed=f, assign=x) for f, x in mine]       # CPU stand-in for bbtn_contract_batch
    e = np.array([bb.BBTN_NEG_INF if r[0] is None else r[0] for r in res], np.int32)
    c = np.array([r[1] & ((1 << 64) - 1) for r in res], np.uint64)
    pe, pc = bb.oplus_combine("mis", e, c)[:2]
    part = torch.tensor([int(pe), int(pc) & 0x7fffffffffffffff, int(pc) >> 63], dtype=torch.int64)
    allp = [torch.zeros(3, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(allp, part)
    ge = np.array([int(p[0]) for p in allp], np.int32)
    gc = np.array([int(p[1]) | (int(p[2]) << 63) for p in allp], np.uint64)
    fe, fc = bb.oplus_combine("mis", ge, gc)[:2]
    # max-over-ranks timing reduction, as bench.py does it
    t = torch.tensor([1.0 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    if rank == 0:
        ref = oracle.frontier_dp(inst)
        with open(out_path, "w") as f:
            json.dump({"got": [int(fe), int(fc)], "ref": [int(ref[0]), int(ref[1])], "leaves": len(leaves),
                       "mine": len(mine), "tmax": float(t[0])}, f)
    h.close()
    dist.destroy_process_group()


def test_leaves_sharded_over_two_ranks_oplus_to_the_unbranched_result(tmp_path):
    import torch.multiprocessing as mp
    out = str(tmp_path / "out.json")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    d = json.load(open(out))
    assert d["got"] == d["ref"] and d["leaves"] > 2 and 0 < d["mine"] < d["leaves"] and d["tmax"] == 2.0


def test_reference_arm_under_torchrun_two_ranks():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--ref-rows", "2", "--ref-leaves", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0
