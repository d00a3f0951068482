// microbench.cu -- register-only integer-pipe microbenchmarks: the measured CUDA-core int32 roof
// that K3 is reported against (include/bbtn.h: bbtn_int32_microbench).
// Many resident warps, 8 independent dependency chains per thread, unrolled, no memory traffic,
// result consumed.  Chains are cross-coupled (Fibonacci-like) so nothing folds to a closed form.
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

constexpr int CH = 8;          // independent chains per thread
constexpr int UNROLL = 16;     // rounds per loop iteration

template <int WHICH>
__global__ void __launch_bounds__(256) pipe_kernel(int iters, int32_t seed, int32_t *sink) {
  int32_t r[CH];
#pragma unroll
  for (int i = 0; i < CH; i++) r[i] = seed * (i + 1) + threadIdx.x;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < UNROLL; u++) {
#pragma unroll
      for (int i = 0; i < CH; i++) {
        const int32_t x = r[(i + 1) % CH], y = r[(i + 3) % CH];
        if (WHICH == 0) asm volatile("add.s32 %0, %0, %1;\n\tadd.s32 %0, %0, %2;" : "+r"(r[i]) : "r"(x), "r"(y));   // -> IADD3
        else if (WHICH == 1) { if (u & 1) asm volatile("max.s32 %0, %0, %1;" : "+r"(r[i]) : "r"(x)); else asm volatile("min.s32 %0, %0, %1;" : "+r"(r[i]) : "r"(y)); }
        else if (WHICH == 2) r[i] = __viaddmax_s32(r[i], x, y);                                                      // max(r+x, y)
        else if (WHICH == 3) asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(x), "r"(y));              // IMAD
        else if (WHICH == 4) {
          if (i & 1) asm volatile("mad.lo.s32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(x), "r"(y));
          else asm volatile("add.s32 %0, %0, %1;\n\tadd.s32 %0, %0, %2;" : "+r"(r[i]) : "r"(x), "r"(y));
        }
      }
    }
  }
  int32_t s = 0;
#pragma unroll
  for (int i = 0; i < CH; i++) s ^= r[i];
  if (s == 0x7fffffff) sink[0] = s;       // consume
}

// per-FMA op mix of the counting GEMM on registers only: an 8x8 register tile, energy pass
// (fused add-max) then count pass (tie test + predicated 64-bit multiply-add).
template <bool WIDE>
__global__ void __launch_bounds__(256) opmix_kernel(int iters, int32_t seed, uint64_t *sink) {
  int32_t ae[8], be[8], acc_e[8][8];
  uint64_t ac[8], bc[8], acc_c[8][8];
#pragma unroll
  for (int i = 0; i < 8; i++) {
    ae[i] = (seed + i * 7 + threadIdx.x) & 63; be[i] = (seed * 3 + i * 5 + threadIdx.x) & 63;
    ac[i] = (uint64_t)(seed + i) | (WIDE ? ((uint64_t)(seed + 2 * i) << 32) : 0);
    bc[i] = (uint64_t)(seed + 3 * i + 1) | (WIDE ? ((uint64_t)(seed + 5 * i) << 32) : 0);
#pragma unroll
    for (int j = 0; j < 8; j++) { acc_e[i][j] = NEG_INF; acc_c[i][j] = 0; }
  }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
      for (int j = 0; j < 8; j++) acc_e[i][j] = __viaddmax_s32(ae[i], be[j], acc_e[i][j]);
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
      for (int j = 0; j < 8; j++) {
        if (ae[i] + be[j] == acc_e[i][j]) {
          if (WIDE) acc_c[i][j] += ac[i] * bc[j];
          else acc_c[i][j] += (uint64_t)(uint32_t)ac[i] * (uint32_t)bc[j];
        }
      }
#pragma unroll
    for (int i = 0; i < 8; i++) { ae[i] = (ae[i] + it) & 63; be[i] = (be[i] ^ it) & 63; }
  }
  uint64_t s = 0;
#pragma unroll
  for (int i = 0; i < 8; i++)
#pragma unroll
    for (int j = 0; j < 8; j++) s += acc_c[i][j] + (uint64_t)acc_e[i][j];
  if (s == 0x123456789abcdefull) sink[0] = s;
}

// two-pipe mixes with two-register operands (fewer register-file reads than the 3-operand mix above):
// WHICH 7: IADD (ALU) : IMAD reg*imm+reg (FMA pipe) = 1:1;  WHICH 8: 2:1.  16 independent chains.
template <int WHICH>
__global__ void __launch_bounds__(256) mix2_kernel(int iters, int32_t seed, int32_t *sink) {
  constexpr int N = 16;
  int32_t r[N];
#pragma unroll
  for (int i = 0; i < N; i++) r[i] = seed * (i + 1) + threadIdx.x;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < 8; u++) {
#pragma unroll
      for (int i = 0; i < N; i++) {
        const bool fma = WHICH == 7 ? (i & 1) : (i % 3 == 2);
        if (fma) asm volatile("mad.lo.s32 %0, %0, 5, %1;" : "+r"(r[i]) : "r"(r[i ^ 2]));
        else asm volatile("add.s32 %0, %0, %1;" : "+r"(r[i]) : "r"(r[i ^ 4]));
      }
    }
  }
  int32_t s = 0;
#pragma unroll
  for (int i = 0; i < N; i++) s ^= r[i];
  if (s == 0x7fffffff) sink[0] = s;
}

// WHICH 9/10: the instruction mix of K3's inner loop on registers only (no operand fetch): per tropical
// FMA one fused add-max into the next-chunk maximum, and add + tie compare + predicated multiply-add
// against the current maximum (gemm_tiled.cu, pass 1 of chunk c+1 interleaved with pass 2 of chunk c).
__global__ void __launch_bounds__(256) k3mix_kernel(int iters, int32_t seed, uint32_t *sink) {
  // operands come from a small shared table read at warp-uniform addresses (one wavefront per LDS.128), so
  // the loop has K3's instruction stream, operand fetches included, without its shared-memory bandwidth
  __shared__ __align__(16) int32_t tab[16][36];
  for (int i = threadIdx.x; i < 16 * 36; i += blockDim.x) tab[i / 36][i % 36] = (i % 36 >= 24) ? 1 + ((seed + i) & 3) : ((seed * 7 + i * 13) & 63);
  __syncthreads();
  int32_t En[4][8], E[4][8]; uint32_t C[4][8];
#pragma unroll
  for (int i = 0; i < 4; i++)
#pragma unroll
    for (int j = 0; j < 8; j++) { En[i][j] = NEG_INF; E[i][j] = 64 + (int)((threadIdx.x + i + j) & 7); C[i][j] = 0; }
  for (int it = 0; it < iters; it++) {
#pragma unroll 4
    for (int kk = 0; kk < 16; kk++) {
      int32_t v[36];
#pragma unroll
      for (int q = 0; q < 9; q++) {
        const int4 x = *reinterpret_cast<const int4 *>(&tab[kk][4 * q]);
        v[4 * q] = x.x; v[4 * q + 1] = x.y; v[4 * q + 2] = x.z; v[4 * q + 3] = x.w;
      }
      // v[0..3] a1, v[4..11] b1, v[12..15] a2, v[16..23] b2, v[24..27] ca, v[28..35] cb
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 8; j++) {
          En[i][j] = __viaddmax_s32(v[i], v[4 + j], En[i][j]);
          asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\tadd.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\t@p mad.lo.u32 %0, %4, %5, %0;\n\t}"
              : "+r"(C[i][j]) : "r"(v[12 + i]), "r"(v[16 + j]), "r"(E[i][j]), "r"(v[24 + i]), "r"(v[28 + j]));
        }
    }
  }
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < 4; i++)
#pragma unroll
    for (int j = 0; j < 8; j++) s += C[i][j] + (uint32_t)En[i][j];
  if (s == 0x12345678u) sink[0] = s;
}

// Issue rates of the instructions the packed and the 64-bit forms of K3 are built from, with operands that change
// every round (nothing can be hoisted): which = 11 VIADDMNMX.S16x2, 12 HSETP2 (+ one SEL that consumes a predicate),
// 13 ISETP (+ SEL), 14 IMAD.WIDE with a 64-bit accumulate, 15 the packed pair of gemm_pack16.cu
// (VIADDMNMX.S16x2 + add + HSETP2 + 2 predicated IMAD = two tropical FMAs).
template <int WHICH>
__global__ void __launch_bounds__(512) pipe2_kernel(int iters, uint32_t seed, uint32_t *sink) {
  uint32_t acc[8], c[8];
#pragma unroll
  for (int i = 0; i < 8; i++) { acc[i] = seed + threadIdx.x * (i + 1); c[i] = seed ^ i; }
  const uint32_t k0 = seed * 7 + threadIdx.x;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < 8; u++) {
#pragma unroll
      for (int i = 0; i < 8; i++) {
        if (WHICH == 11) acc[i] = __viaddmax_s16x2(acc[(i + 1) & 7], k0, acc[i]);
        else if (WHICH == 12) asm volatile("{.reg .pred p,q; setp.eq.f16x2 p|q, %0, %1; selp.u32 %0, %1, %2, p; }" : "+r"(acc[i]) : "r"(acc[(i + 1) & 7]), "r"(k0));
        else if (WHICH == 13) asm volatile("{.reg .pred p; setp.eq.s32 p, %0, %1; selp.u32 %0, %1, %2, p; }" : "+r"(acc[i]) : "r"(acc[(i + 1) & 7]), "r"(k0));
        else if (WHICH == 14) {
          unsigned long long w = ((unsigned long long)c[i] << 32) | acc[i];
          asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(w) : "r"(acc[(i + 1) & 7]), "r"(k0));
          acc[i] = (uint32_t)w; c[i] = (uint32_t)(w >> 32);
        } else {
          uint32_t s;
          acc[i] = __viaddmax_s16x2(acc[(i + 1) & 7], k0, acc[i]);
          asm volatile("{.reg .pred p,q; add.u32 %2, %3, %4; setp.eq.f16x2 p|q, %2, %5; @p mad.lo.u32 %0, %3, %4, %0; @q mad.lo.u32 %1, %4, %4, %1;}"
                       : "+r"(c[i]), "+r"(c[(i + 4) & 7]), "=r"(s) : "r"(acc[(i + 2) & 7]), "r"(k0), "r"(acc[i]));
        }
      }
    }
  }
  uint32_t r = 0;
#pragma unroll
  for (int i = 0; i < 8; i++) r += c[i] ^ acc[i];
  if (r == 0x12345678u) sink[0] = r;
}

}  // namespace

int run_microbench(int which, int iters, double *ms, double *ops, cudaStream_t st) {
  void *sink = nullptr;
  if (cudaMalloc(&sink, 64) != cudaSuccess) return 3;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  int grid = 148 * 8, block = 256;
  if (which == 9) { grid = 148; block = 256; }          // 2 warps per SM sub-partition, as K3 runs
  if (which == 10) { grid = 148 * 4; block = 256; }     // same mix, 4+ warps per sub-partition
  if (which >= 11) { grid = 148 * 4; block = 512; }
  auto launch = [&](int n) {
    switch (which) {
      case 7: mix2_kernel<7><<<grid, block, 0, st>>>(n, 12345, (int32_t *)sink); break;
      case 8: mix2_kernel<8><<<grid, block, 0, st>>>(n, 12345, (int32_t *)sink); break;
      case 9: case 10: k3mix_kernel<<<grid, block, 0, st>>>(n, 12345, (uint32_t *)sink); break;
      case 0: pipe_kernel<0><<<grid, block, 0, st>>>(n, 12345, (int32_t *)sink); break;
      case 1: pipe_kernel<1><<<grid, block, 0, st>>>(n, 12345, (int32_t *)sink); break;
      case 2: pipe_kernel<2><<<grid, block, 0, st>>>(n, 12345, (int32_t *)sink); break;
      case 3: pipe_kernel<3><<<grid, block, 0, st>>>(n, 12345, (int32_t *)sink); break;
      case 4: pipe_kernel<4><<<grid, block, 0, st>>>(n, 12345, (int32_t *)sink); break;
      case 11: pipe2_kernel<11><<<grid, block, 0, st>>>(n, 12345u, (uint32_t *)sink); break;
      case 12: pipe2_kernel<12><<<grid, block, 0, st>>>(n, 12345u, (uint32_t *)sink); break;
      case 13: pipe2_kernel<13><<<grid, block, 0, st>>>(n, 12345u, (uint32_t *)sink); break;
      case 14: pipe2_kernel<14><<<grid, block, 0, st>>>(n, 12345u, (uint32_t *)sink); break;
      case 15: pipe2_kernel<15><<<grid, block, 0, st>>>(n, 12345u, (uint32_t *)sink); break;
      case 5: opmix_kernel<true><<<grid, block, 0, st>>>(n, 12345, (uint64_t *)sink); break;
      default: opmix_kernel<false><<<grid, block, 0, st>>>(n, 12345, (uint64_t *)sink); break;
    }
  };
  launch(iters / 8 + 1);                       // warm-up
  cudaEventRecord(e0, st);
  launch(iters);
  cudaEventRecord(e1, st);
  cudaError_t err = cudaEventSynchronize(e1);
  float t = 0;
  cudaEventElapsedTime(&t, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(sink);
  if (err != cudaSuccess || cudaGetLastError() != cudaSuccess) return 3;
  *ms = t;
  const double threads = (double)grid * block;
  if (which <= 4) {
    double per_round = CH;                     // one instruction per chain per round
    *ops = threads * (double)iters * UNROLL * per_round;
  } else if (which == 7 || which == 8) {
    *ops = threads * (double)iters * 8.0 * 16.0;   // lane-instructions
  } else if (which == 9 || which == 10) {
    *ops = threads * (double)iters * 16.0 * 32.0;   // tropical FMAs (4 instructions each + 9 LDS.128 per 32)
  } else if (which >= 11) {
    *ops = threads * (double)iters * 64.0;          // rounds: one instruction (11, 14), one compare + SEL (12, 13), one packed pair (15)
  } else {
    *ops = threads * (double)iters * 64.0;     // tropical FMAs
  }
  return 0;
}

}  // namespace bbtn
