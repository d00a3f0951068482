// gemm.cu -- K3: register- and shared-memory-tiled batched counting-tropical GEMM (sm_100a).
//
//   C[b,g,m,n] = (+)_k A[b,g,m,k] (.) B[b,g,k,n]        (PAPER.md:51 Eq. 2 evaluated pairwise, :57)
//   (ea,ca) (.) (eb,cb) = (ea+eb, ca*cb);  (+) keeps the max energy, adds counts on ties.
//
// Tensor cores cannot evaluate max-plus, so this runs on the integer CUDA cores (north_star).
// v1: single pass, 64x64 CTA tile, BK = 16, 256 threads, 4x4 outputs per thread.
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

constexpr int BM = 64, BN = 64, BK = 16, TM = 4, TN = 4, NT = 256;

// c += (ea + eb == E) ? lo32(ca) * lo32(cb) : 0, as SEL + IMAD.WIDE with the 64-bit accumulate fused
template <class CT>
__device__ __forceinline__ void tie_fma_narrow(CT &c, int32_t ea, int32_t eb, int32_t E, CT ca, CT cb) {
  uint64_t c64 = (uint64_t)c;
  asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\t.reg .u32 t;\n\tadd.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\t"
      "selp.u32 t, %5, 0, p;\n\tmad.wide.u32 %0, %4, t, %0;\n\t}"
      : "+l"(c64) : "r"(ea), "r"(eb), "r"(E), "r"((uint32_t)ca), "r"((uint32_t)cb));
  c = (CT)c64;
}

// NARROW: both operands' counts are < 2^32 (caller's count_bits <= 32, RING_U64 only), so the
// product is one 32x32->64 multiply instead of a 64x64->64 one; the result is the same number.
template <class R, bool A_KMAJOR, bool NARROW = false>
__global__ void __launch_bounds__(NT, NARROW ? 2 : 1) gemm_tiled_kernel(int64_t G, int M, int N, int K,
                                                        const int32_t *__restrict__ Ae, const typename R::T *__restrict__ Ac,
                                                        const int32_t *__restrict__ Be, const typename R::T *__restrict__ Bc,
                                                        int32_t *__restrict__ Ce, typename R::T *__restrict__ Cc,
                                                        int64_t sA, int64_t sB, int64_t sC) {
  using CT = typename R::T;
  __shared__ int32_t As_e[BK][BM + 4];
  __shared__ CT As_c[BK][BM + 2];
  __shared__ int32_t Bs_e[BK][BN + 4];
  __shared__ CT Bs_c[BK][BN + 2];

  const int tiles_n = (N + BN - 1) / BN, tiles_m = (M + BM - 1) / BM;
  const int64_t bg = blockIdx.x / (tiles_n * tiles_m);
  const int tile = (int)(blockIdx.x - bg * (tiles_n * tiles_m));
  const int64_t b = bg / G, g = bg - b * G;
  const int m0 = (tile / tiles_n) * BM, n0 = (tile % tiles_n) * BN;
  const int32_t *ae = Ae + b * sA + g * (int64_t)M * K; const CT *ac = Ac + b * sA + g * (int64_t)M * K;
  const int32_t *be = Be + b * sB + g * (int64_t)K * N; const CT *bc = Bc + b * sB + g * (int64_t)K * N;
  int32_t *ce = Ce + b * sC + g * (int64_t)M * N; CT *cc = Cc + b * sC + g * (int64_t)M * N;

  const int tx = threadIdx.x % (BN / TN), ty = threadIdx.x / (BN / TN);   // 16 x 16 threads
  int32_t acc_e[TM][TN]; CT acc_c[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; i++)
#pragma unroll
    for (int j = 0; j < TN; j++) { acc_e[i][j] = NEG_INF; acc_c[i][j] = 0; }

  for (int k0 = 0; k0 < K; k0 += BK) {
    // stage A tile as [k][m] and B tile as [k][n]; out-of-range entries are the zero element
    for (int i = threadIdx.x; i < BM * BK; i += NT) {
      int kk, mm;
      if (A_KMAJOR) { kk = i / BM; mm = i % BM; } else { mm = i / BK; kk = i % BK; }
      const int gm = m0 + mm, gk = k0 + kk;
      int32_t e = NEG_INF; CT c = 0;
      if (gm < M && gk < K) {
        const int64_t idx = A_KMAJOR ? (int64_t)gk * M + gm : (int64_t)gm * K + gk;
        e = ae[idx]; c = ac[idx];
      }
      As_e[kk][mm] = e; As_c[kk][mm] = c;
    }
    for (int i = threadIdx.x; i < BN * BK; i += NT) {
      const int kk = i / BN, nn = i % BN;
      const int gn = n0 + nn, gk = k0 + kk;
      int32_t e = NEG_INF; CT c = 0;
      if (gn < N && gk < K) { e = be[(int64_t)gk * N + gn]; c = bc[(int64_t)gk * N + gn]; }
      Bs_e[kk][nn] = e; Bs_c[kk][nn] = c;
    }
    __syncthreads();
    if (NARROW) {
      // two passes over the chunk, as in gemm_tiled.cu: (1) the running maximum, one fused add-max per term;
      // (2) where it rose the old count is dropped, then every term that ties with it adds its product
      // (compare + select + 32x32+64 multiply-add).  ~5 integer instructions per term instead of ~12.
      int32_t new_e[TM][TN];
#pragma unroll
      for (int i = 0; i < TM; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) new_e[i][j] = acc_e[i][j];
#pragma unroll 2
      for (int kk = 0; kk < BK; kk++) {
        int32_t a_e[TM], b_e[TN];
#pragma unroll
        for (int i = 0; i < TM; i++) a_e[i] = As_e[kk][ty * TM + i];
#pragma unroll
        for (int j = 0; j < TN; j++) b_e[j] = Bs_e[kk][tx * TN + j];
#pragma unroll
        for (int i = 0; i < TM; i++)
#pragma unroll
          for (int j = 0; j < TN; j++) new_e[i][j] = max(new_e[i][j], a_e[i] + b_e[j]);
      }
#pragma unroll
      for (int i = 0; i < TM; i++)
#pragma unroll
        for (int j = 0; j < TN; j++)
          if (new_e[i][j] > acc_e[i][j]) { acc_e[i][j] = new_e[i][j]; acc_c[i][j] = 0; }
#pragma unroll 2
      for (int kk = 0; kk < BK; kk++) {
        int32_t a_e[TM], b_e[TN]; CT a_c[TM], b_c[TN];
#pragma unroll
        for (int i = 0; i < TM; i++) { a_e[i] = As_e[kk][ty * TM + i]; a_c[i] = As_c[kk][ty * TM + i]; }
#pragma unroll
        for (int j = 0; j < TN; j++) { b_e[j] = Bs_e[kk][tx * TN + j]; b_c[j] = Bs_c[kk][tx * TN + j]; }
#pragma unroll
        for (int i = 0; i < TM; i++)
#pragma unroll
          for (int j = 0; j < TN; j++) tie_fma_narrow(acc_c[i][j], a_e[i], b_e[j], acc_e[i][j], a_c[i], b_c[j]);
      }
    } else {
#pragma unroll
    for (int kk = 0; kk < BK; kk++) {
      int32_t a_e[TM], b_e[TN]; CT a_c[TM], b_c[TN];
#pragma unroll
      for (int i = 0; i < TM; i++) { a_e[i] = As_e[kk][ty * TM + i]; a_c[i] = As_c[kk][ty * TM + i]; }
#pragma unroll
      for (int j = 0; j < TN; j++) { b_e[j] = Bs_e[kk][tx * TN + j]; b_c[j] = Bs_c[kk][tx * TN + j]; }
#pragma unroll
      for (int i = 0; i < TM; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) oplus<R>(acc_e[i][j], acc_c[i][j], a_e[i] + b_e[j],
                   NARROW ? (CT)((uint64_t)(uint32_t)a_c[i] * (uint32_t)b_c[j]) : R::mul(a_c[i], b_c[j]));
    }
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < TM; i++)
#pragma unroll
    for (int j = 0; j < TN; j++) {
      const int gm = m0 + ty * TM + i, gn = n0 + tx * TN + j;
      if (gm < M && gn < N) {
        int32_t e = acc_e[i][j]; CT c = acc_c[i][j];
        canonicalise<R>(e, c);
        ce[(int64_t)gm * N + gn] = e; cc[(int64_t)gm * N + gn] = c;
      }
    }
}

}  // namespace

void launch_gemm_tiled(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                       const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc, int32_t *Ce, void *Cc,
                       int64_t sA, int64_t sB, int64_t sC, int ring, int count_bits, cudaStream_t st) {
  // RING_U64 runs on the 128-row streaming tile of gemm_tiled.cu, except where that tile would be
  // >= 75 % padding (M, N <= 64): there the 64x64 tile below wastes nothing and many CTAs fit per SM.
  if (ring == RING_U64 && !(M <= BM && N <= BN)) {
    launch_gemm_tiled_u64(batch, G, M, N, K, a_kmajor, Ae, (const uint64_t *)Ac, Be, (const uint64_t *)Bc, Ce, (uint64_t *)Cc,
                          sA, sB, sC, count_bits, st);
    return;
  }
  const int64_t n_cta = (int64_t)((N + BN - 1) / BN) * ((M + BM - 1) / BM) * batch * G;
  dim3 grid((unsigned)n_cta);
  if (ring == RING_U64 && count_bits <= 32) {
    using R = RingU64;
    const uint64_t *ac = (const uint64_t *)Ac, *bc = (const uint64_t *)Bc; uint64_t *cc = (uint64_t *)Cc;
    if (a_kmajor) gemm_tiled_kernel<R, true, true><<<grid, NT, 0, st>>>(G, M, N, K, Ae, ac, Be, bc, Ce, cc, sA, sB, sC);
    else gemm_tiled_kernel<R, false, true><<<grid, NT, 0, st>>>(G, M, N, K, Ae, ac, Be, bc, Ce, cc, sA, sB, sC);
    return;
  }
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    if (a_kmajor)
      gemm_tiled_kernel<R, true><<<grid, NT, 0, st>>>(G, M, N, K, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc, sA, sB, sC);
    else
      gemm_tiled_kernel<R, false><<<grid, NT, 0, st>>>(G, M, N, K, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc, sA, sB, sC);
  });
}

}  // namespace bbtn
