// gemm.cu -- K3: register- and shared-memory-tiled batched counting-tropical GEMM (sm_100a).
//
//   C[b,g,m,n] = (+)_k A[b,g,m,k] (.) B[b,g,k,n]        (PAPER.md:51 Eq. 2 evaluated pairwise, :57)
//   (ea,ca) (.) (eb,cb) = (ea+eb, ca*cb);  (+) keeps the max energy, adds counts on ties.
//
// Tensor cores cannot evaluate max-plus, so this runs on the integer CUDA cores (north_star).
// 64x64 CTA tile, BK = 16, 256 threads, 4x4 outputs per thread, two cp.async-fed shared-memory stages.
// Used by the mod-p rings and by RING_U64 shapes with M, N <= 64 (gemm_tiled.cu has the 128-row tile).
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

constexpr int BM = 64, BN = 64, BK = 16, TM = 4, TN = 4, NT = 256;

template <class CT> struct Stage {
  static constexpr int AE = 0, AC = AE + BK * (BM + 4) * 4, BE = AC + BK * (BM + 2) * (int)sizeof(CT),
                       BC = BE + BK * (BN + 4) * 4, BYTES = BC + BK * (BN + 2) * (int)sizeof(CT);
  static_assert(AC % 8 == 0 && BE % 8 == 0 && BC % 8 == 0 && BYTES % 16 == 0, "stage alignment");
};

// 4- or 8-byte asynchronous global -> shared copy (element-wise: the A tile is transposed on the way in)
template <int BYTES> __device__ __forceinline__ void cp_async_small(void *smem, const void *gmem) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(d), "l"(gmem), "n"(BYTES) : "memory");
}

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
  // two stages, each [k][m] A energies / counts and [k][n] B energies / counts; the next chunk is
  // brought in by cp.async while the current one is consumed (no staging registers)
  using S = Stage<CT>;
  extern __shared__ __align__(16) unsigned char dsm[];

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

  // stage A tile as [k][m] and B tile as [k][n]; out-of-range entries are the zero element
  auto fill = [&](int st, int k0) {
    unsigned char *base = dsm + st * S::BYTES;
    auto Ase = reinterpret_cast<int32_t (*)[BM + 4]>(base + S::AE); auto Asc = reinterpret_cast<CT (*)[BM + 2]>(base + S::AC);
    auto Bse = reinterpret_cast<int32_t (*)[BN + 4]>(base + S::BE); auto Bsc = reinterpret_cast<CT (*)[BN + 2]>(base + S::BC);
    for (int i = threadIdx.x; i < BM * BK; i += NT) {
      int kk, mm;
      if (A_KMAJOR) { kk = i / BM; mm = i % BM; } else { mm = i / BK; kk = i % BK; }
      const int gm = m0 + mm, gk = k0 + kk;
      if (gm < M && gk < K) {
        const int64_t idx = A_KMAJOR ? (int64_t)gk * M + gm : (int64_t)gm * K + gk;
        cp_async_small<4>(&Ase[kk][mm], ae + idx); cp_async_small<(int)sizeof(CT)>(&Asc[kk][mm], ac + idx);
      } else { Ase[kk][mm] = NEG_INF; Asc[kk][mm] = 0; }
    }
    for (int i = threadIdx.x; i < BN * BK; i += NT) {
      const int kk = i / BN, nn = i % BN;
      const int gn = n0 + nn, gk = k0 + kk;
      if (gn < N && gk < K) {
        const int64_t idx = (int64_t)gk * N + gn;
        cp_async_small<4>(&Bse[kk][nn], be + idx); cp_async_small<(int)sizeof(CT)>(&Bsc[kk][nn], bc + idx);
      } else { Bse[kk][nn] = NEG_INF; Bsc[kk][nn] = 0; }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  fill(0, 0);
  for (int k0 = 0, chunk = 0; k0 < K; k0 += BK, chunk++) {
    const int cur = chunk & 1;
    if (k0 + BK < K) { fill(cur ^ 1, k0 + BK); asm volatile("cp.async.wait_group 1;" ::: "memory"); }
    else asm volatile("cp.async.wait_group 0;" ::: "memory");
    unsigned char *base = dsm + cur * S::BYTES;
    auto As_e = reinterpret_cast<int32_t (*)[BM + 4]>(base + S::AE); auto As_c = reinterpret_cast<CT (*)[BM + 2]>(base + S::AC);
    auto Bs_e = reinterpret_cast<int32_t (*)[BN + 4]>(base + S::BE); auto Bs_c = reinterpret_cast<CT (*)[BN + 2]>(base + S::BC);
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

template <class R, bool A_KMAJOR, bool NARROW>
void launch_v1(dim3 grid, cudaStream_t st, int64_t G, int M, int N, int K, const int32_t *Ae, const typename R::T *Ac,
               const int32_t *Be, const typename R::T *Bc, int32_t *Ce, typename R::T *Cc, int64_t sA, int64_t sB, int64_t sC) {
  constexpr int SMEM = 2 * Stage<typename R::T>::BYTES;
  // per function AND per device, so set it on every launch (a cheap host-side call)
  cudaFuncSetAttribute(gemm_tiled_kernel<R, A_KMAJOR, NARROW>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
  gemm_tiled_kernel<R, A_KMAJOR, NARROW><<<grid, NT, SMEM, st>>>(G, M, N, K, Ae, Ac, Be, Bc, Ce, Cc, sA, sB, sC);
}

}  // namespace

void launch_gemm_tiled(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                       const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc, int32_t *Ce, void *Cc,
                       int64_t sA, int64_t sB, int64_t sC, int ring, int count_bits, int energy_bits, cudaStream_t st) {
  if (ring == RING_NONE) {                                 // search mode: the energy plane alone (gemm_maxplus.cu)
    launch_gemm_maxplus(batch, G, M, N, K, a_kmajor, Ae, Be, Ce, sA, sB, sC, energy_bits, st);
    return;
  }
  // RING_U64 runs on the 128-row streaming tile of gemm_tiled.cu, except where that tile would be
  // >= 75 % padding (M, N <= 64): there the 64x64 tile below wastes nothing and many CTAs fit per SM.
  if (ring == RING_U64 && (!(M <= BM && N <= BN) || gemm_pack16_eligible(K, count_bits, energy_bits))) {
    launch_gemm_tiled_u64(batch, G, M, N, K, a_kmajor, Ae, (const uint64_t *)Ac, Be, (const uint64_t *)Bc, Ce, (uint64_t *)Cc,
                          sA, sB, sC, count_bits, energy_bits, st);
    return;
  }
  const int64_t n_cta = (int64_t)((N + BN - 1) / BN) * ((M + BM - 1) / BM) * batch * G;
  dim3 grid((unsigned)n_cta);
  if (ring == RING_U64 && count_bits <= 32) {
    using R = RingU64;
    const uint64_t *ac = (const uint64_t *)Ac, *bc = (const uint64_t *)Bc; uint64_t *cc = (uint64_t *)Cc;
    if (a_kmajor) launch_v1<R, true, true>(grid, st, G, M, N, K, Ae, ac, Be, bc, Ce, cc, sA, sB, sC);
    else launch_v1<R, false, true>(grid, st, G, M, N, K, Ae, ac, Be, bc, Ce, cc, sA, sB, sC);
    return;
  }
  if (ring == RING_P12) {                                  // both prime residues packed in one 64-bit count (CRT mode's second pass)
    using R = RingP12;
    const uint64_t *ac = (const uint64_t *)Ac, *bc = (const uint64_t *)Bc; uint64_t *cc = (uint64_t *)Cc;
    if (a_kmajor) launch_v1<R, true, false>(grid, st, G, M, N, K, Ae, ac, Be, bc, Ce, cc, sA, sB, sC);
    else launch_v1<R, false, false>(grid, st, G, M, N, K, Ae, ac, Be, bc, Ce, cc, sA, sB, sC);
    return;
  }
  {                                                        // RING_U64 with full-width counts on a small matrix
    using R = RingU64;
    using CT = typename R::T;
    if (a_kmajor)
      launch_v1<R, true, false>(grid, st, G, M, N, K, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc, sA, sB, sC);
    else
      launch_v1<R, false, false>(grid, st, G, M, N, K, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc, sA, sB, sC);
  }
}

}  // namespace bbtn
