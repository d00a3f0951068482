// gemm_stage.cuh -- operand staging shared by the tiled K3 kernels (gemm_tiled.cu, gemm_pack16.cu):
// tile constants, launch arguments, cp.async helpers and the global -> shared fill of one K-chunk.
#pragma once
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace stage {

constexpr int BM = 128, BK = 16, NT = 256;   // NT: threads of the 32-bit kernels (the fill functions take it as a parameter)
constexpr int RAW_STAGES = 2, CONV_STAGES = 3;
constexpr int AE_LD = BK + 4;            // row-major A energies: [BM][AE_LD] int32 (row stride 80 B)
constexpr int AC_LD = BK + 2;            // row-major A counts:   [BM][AC_LD] uint64 (row stride 144 B)
constexpr int AE_BYTES = BM * AE_LD * 4; // k-major A needs BK*BM*4 <= this
constexpr int AC_BYTES = BM * AC_LD * 8;

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct GemmArgs {
  int64_t G;
  int M, N, K;
  const int32_t *Ae; const uint64_t *Ac; const int32_t *Be; const uint64_t *Bc;
  int32_t *Ce; uint64_t *Cc;
  int64_t sA, sB, sC;
  int vecA, vecB, vecC;     // 16-byte paths allowed (alignment of pointers, strides and leading dimensions)
};

// ---- global -> shared for one chunk (k0 .. k0+BK) of one operand ------------------------------
template <bool A_KMAJOR, int NT = 256, int TBM = 128>
__device__ __forceinline__ void fill_A(const GemmArgs &p, const int32_t *__restrict__ ae, const uint64_t *__restrict__ ac,
                                       int m0, int k0, unsigned char *sAe, unsigned char *sAc) {
  constexpr int BM = TBM;                 // rows of the A tile (the 64-row packed kernel uses a smaller tile)
  const int t = threadIdx.x;
  const bool fast = p.vecA && m0 + BM <= p.M && k0 + BK <= p.K;
  if (fast) {
    if (A_KMAJOR) {
#pragma unroll
      for (int idx = t; idx < BK * BM / 4; idx += NT) {
        const int kk = idx / (BM / 4), q = idx % (BM / 4);
        cp_async16(sAe + (kk * BM + 4 * q) * 4, ae + (int64_t)(k0 + kk) * p.M + m0 + 4 * q);
      }
#pragma unroll
      for (int idx = t; idx < BK * BM / 2; idx += NT) {
        const int kk = idx / (BM / 2), q = idx % (BM / 2);
        cp_async16(sAc + (kk * BM + 2 * q) * 8, ac + (int64_t)(k0 + kk) * p.M + m0 + 2 * q);
      }
    } else {
#pragma unroll
      for (int idx = t; idx < BM * BK / 4; idx += NT) {
        const int r = idx / (BK / 4), q = idx % (BK / 4);
        cp_async16(sAe + (r * AE_LD + 4 * q) * 4, ae + (int64_t)(m0 + r) * p.K + k0 + 4 * q);
      }
#pragma unroll
      for (int idx = t; idx < BM * BK / 2; idx += NT) {
        const int r = idx / (BK / 2), q = idx % (BK / 2);
        cp_async16(sAc + (r * AC_LD + 2 * q) * 8, ac + (int64_t)(m0 + r) * p.K + k0 + 2 * q);
      }
    }
  } else {
    int32_t *se = reinterpret_cast<int32_t *>(sAe);
    uint64_t *sc = reinterpret_cast<uint64_t *>(sAc);
    for (int idx = t; idx < BM * BK; idx += NT) {
      int r, kk;
      if (A_KMAJOR) { kk = idx / BM; r = idx % BM; } else { r = idx / BK; kk = idx % BK; }
      const int gm = m0 + r, gk = k0 + kk;
      int32_t e = NEG_INF; uint64_t c = 0;
      if (gm < p.M && gk < p.K) {
        const int64_t gi = A_KMAJOR ? (int64_t)gk * p.M + gm : (int64_t)gm * p.K + gk;
        e = ae[gi]; c = ac[gi];
      }
      if (A_KMAJOR) { se[kk * BM + r] = e; sc[kk * BM + r] = c; }
      else { se[r * AE_LD + kk] = e; sc[r * AC_LD + kk] = c; }
    }
  }
}

template <int BNt, int NT = 256>
__device__ __forceinline__ void fill_B(const GemmArgs &p, const int32_t *__restrict__ be, const uint64_t *__restrict__ bc,
                                       int n0, int k0, unsigned char *sBe, unsigned char *sBc) {
  const int t = threadIdx.x;
  const bool fast = p.vecB && n0 + BNt <= p.N && k0 + BK <= p.K;
  if (fast) {
#pragma unroll
    for (int idx = t; idx < BK * BNt / 4; idx += NT) {
      const int kk = idx / (BNt / 4), q = idx % (BNt / 4);
      cp_async16(sBe + (kk * BNt + 4 * q) * 4, be + (int64_t)(k0 + kk) * p.N + n0 + 4 * q);
    }
#pragma unroll
    for (int idx = t; idx < BK * BNt / 2; idx += NT) {
      const int kk = idx / (BNt / 2), q = idx % (BNt / 2);
      cp_async16(sBc + (kk * (BNt / 2) + q) * 16, bc + (int64_t)(k0 + kk) * p.N + n0 + 2 * q);
    }
  } else {
    int32_t *se = reinterpret_cast<int32_t *>(sBe);
    uint64_t *sc = reinterpret_cast<uint64_t *>(sBc);
    for (int idx = t; idx < BK * BNt; idx += NT) {
      const int kk = idx / BNt, n = idx % BNt;
      const int gn = n0 + n, gk = k0 + kk;
      int32_t e = NEG_INF; uint64_t c = 0;
      if (gn < p.N && gk < p.K) { e = be[(int64_t)gk * p.N + gn]; c = bc[(int64_t)gk * p.N + gn]; }
      se[kk * BNt + n] = e;
      sc[kk * BNt + n] = c;
    }
  }
}

}  // namespace stage
}  // namespace bbtn
