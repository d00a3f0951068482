"""Raw batched counting-tropical GEMM sweep (BASELINE.json configs[3], first half), through the C ABI.

    python -m paper_2602_05470_b200.gemm_sweep [--sizes 64 256 1024 4096] [--batches 1 4 16 64 256 1024] [--modes 3:7 3:32 14:32 32:32 64:32]

M = N = K = n, energies uniform in [-64, 64], counts uniform in {1..4} (instances.gemm_operands); batches are
restricted to B * 3 * n^2 * 12 B <= --max-gb.  One JSON line per (n, B, count_bits): milliseconds (CUDA events,
median of --repeat after 2 warm-ups), GFMA/s (1 tropical FMA = one (b, m, n, k) term) and Gop/s = 2 x GFMA/s.
A mode is count_bits:energy_bits, the caller's promises on the operands (include/bbtn.h): 3:7 selects the packed
16x2 form (small counts and |energy| < 2^7), 3:32 32-bit energies with 32-bit accumulators, 14:32 chunk-local
32-bit tie sums with 64-bit accumulators, 32:32 32-bit operands with 64-bit accumulators, 64:32 the full 64x64 multiply.
13:7 and 32:7 are the packed form with 64-bit totals (carry form for counts < 2^13; 64-bit accumulators for counts < 2^32).
count_bits 0 is the search mode's K3 (bbtn_maxplus_gemm_batched: energy planes alone, 4 B per element): 0:7 its packed
16-bit form, 0:32 its 32-bit form.
"""
from __future__ import annotations

import argparse
import json

import numpy as np

from . import binding as bb
from . import instances as I


def main():
    import torch
    ap = argparse.ArgumentParser()
    ap.add_argument("--sizes", nargs="*", type=int, default=[64, 256, 1024, 4096])
    ap.add_argument("--batches", nargs="*", type=int, default=[1, 4, 16, 64, 256, 1024])
    ap.add_argument("--modes", nargs="*", default=["3:7", "3:32", "14:32", "32:32", "64:32"])
    ap.add_argument("--max-gb", type=float, default=16.0)
    ap.add_argument("--repeat", type=int, default=5)
    a = ap.parse_args()
    bb.load()
    st = torch.cuda.Stream()
    for n in a.sizes:
        for B in a.batches:
            if B * 3.0 * n * n * 12 > a.max_gb * 1e9:
                continue
            # one seeded entry is generated per (n, B) up to 8 entries and tiled over the batch (values repeat, shapes do not)
            gen = min(B, 8)
            Ae, Ac, Be, Bc = I.gemm_operands(gen, n, n, n, seed=1000 * n + B)
            rep = lambda x: torch.from_numpy(x.view(np.int64) if x.dtype == np.uint64 else x).cuda().repeat((B + gen - 1) // gen, 1, 1)[:B].contiguous()
            dAe, dAc, dBe, dBc = rep(Ae), rep(Ac), rep(Be), rep(Bc)
            dCe = torch.empty((B, n, n), dtype=torch.int32, device="cuda"); dCc = torch.empty((B, n, n), dtype=torch.int64, device="cuda")
            for mode in a.modes:
                bits, ebits = (int(x) for x in mode.split(":"))
                if bits == 0:
                    run = lambda: bb.maxplus_gemm_batched(dAe, dBe, dCe, energy_bits=ebits, stream=st.cuda_stream)
                else:
                    run = lambda: bb.tropical_gemm_batched(dAe, dAc, dBe, dBc, dCe, dCc, count_bits=bits, energy_bits=ebits, stream=st.cuda_stream)
                with torch.cuda.stream(st):
                    for _ in range(2):
                        run()
                    ts = []
                    for _ in range(a.repeat):
                        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                        e0.record(st)
                        run()
                        e1.record(st); e1.synchronize()
                        ts.append(e0.elapsed_time(e1))
                ms = float(np.median(ts))
                fma = float(B) * n * n * n
                print(json.dumps({"n": n, "batch": B, "count_bits": bits, "energy_bits": ebits, "ms": ms, "gfma_per_s": fma / ms / 1e6,
                                  "gop_per_s": 2 * fma / ms / 1e6, "bytes": B * 3 * n * n * (12 if bits else 4)}), flush=True)
            del dAe, dAc, dBe, dBc, dCe, dCc


if __name__ == "__main__":
    main()
