// gemm_maxplus.cu -- K3 in SEARCH mode: batched max-plus GEMM on the energy plane alone.
//
//   C[b,g,m,n] = max_k ( A[b,g,m,k] + B[b,g,k,n] )         (PAPER.md:51 Eq. 2 evaluated pairwise, :57, in the
//                                                            semiring without counts: "the tropical
//                                                            number inf for optimization problems", :81-91)
//
// One fused add-max per tropical FMA and nothing else in the inner loop:
//   * 16-bit form (caller promises |e| < 2^11 for every finite energy, the zero element exactly BBTN_NEG_INF):
//     energies are encoded as enc(e) = e + BIAS (zero element -> 0) in 16-bit halves, two neighbouring output
//     columns share one register and one VIADDMNMX.S16x2 does TWO tropical FMAs.  A finite + finite sum is
//     >= 2 (BIAS - 3967) = FINITE2 and every sum that involves a zero element stays below it, so the decode
//     of the final maximum tells the two apart (the encoding argument of gemm_pack16.cu);
//   * 32-bit form (any energy within +-BBTN_ENERGY_LIMIT): one VIADDMNMX per FMA; -2^30 + -2^30 = INT_MIN does
//     not overflow and every sum with a zero element is below ZERO_BELOW: canonicalised to BBTN_NEG_INF on store.
// Tile TB x TB (128, or 64 for matrices with M, N <= 64), 8 x 8 outputs per thread, TB*TB/64 threads.  Operands go
// global -> registers -> shared memory (encoded once, A k-major: a row-major A is transposed on the way, with an
// XOR swizzle of the row index that keeps both the transposing stores and the 16-byte reads conflict-free),
// double-buffered: the loads of chunk c+1 are in flight while chunk c is computed, one barrier per chunk.
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

constexpr int BIAS = 11903, FINITE2 = 15872;   // enc(e) = e + BIAS;  half >= FINITE2  <=>  finite sum

struct MpArgs {
  int64_t G;
  int M, N, K;
  const int32_t *A, *B;
  int32_t *C;
  int64_t sA, sB, sC;
  int vecA, vecB, vecC;     // 16-byte paths allowed (alignment of pointers, strides and leading dimensions)
};

template <bool P16, int TB> struct Cfg {
  static constexpr int NT = TB * TB / 64;                       // 8 x 8 outputs per thread
  static constexpr int BK = (P16 && TB == 128) ? 32 : 16;
  static constexpr int BW = P16 ? TB / 2 : TB;                  // 32-bit words per k-row of the B stage
  static constexpr int UNITS = (TB * BK / 4) / NT;              // 16-byte global loads per thread, chunk and operand
  static constexpr int SWZ = 128 / BK;                          // row-major A: row ^= (k / 4) * SWZ, a multiple of 4
  static constexpr int STAGE_WORDS = BK * TB + BK * BW;
  static_assert(UNITS >= 1 && (TB * BK / 4) % NT == 0, "fill mapping");
  static_assert(2 * STAGE_WORDS * 4 <= 48 * 1024, "static shared memory");
};

// enc(e) = max(e + BIAS, 0): a finite e >= -3967 gives e + BIAS > 0, any zero element (e < -2^29) a negative sum -> 0;
// one VIADDMNMX instead of compare + add + select (the encoders run on the same ALU pipe as the FMAs)
__device__ __forceinline__ uint32_t enc16(int32_t e) { return (uint32_t)__viaddmax_s32(e, BIAS, 0); }
__device__ __forceinline__ uint32_t canon32(int32_t e) { return (uint32_t)(e < ZERO_BELOW ? NEG_INF : e); }   // non-canonical zero -> canonical
template <bool P16> __device__ __forceinline__ uint32_t enc_a(int32_t e) {
  if (P16) return enc16(e) * 0x10001u;                                        // the value in both halves
  return canon32(e);
}
// two encoded halves in one word; written as a multiply-add so that it issues on the FMA pipe (IMAD), not the ALU pipe
__device__ __forceinline__ uint32_t pack2(int32_t lo, int32_t hi) { return enc16(hi) * 0x10000u + enc16(lo); }

__device__ __forceinline__ void lds4(const uint32_t *src, uint32_t *dst) {
  const uint4 v = *reinterpret_cast<const uint4 *>(src);
  dst[0] = v.x; dst[1] = v.y; dst[2] = v.z; dst[3] = v.w;
}

template <bool A_KMAJOR, bool P16, int TB>
__global__ void __launch_bounds__(Cfg<P16, TB>::NT, TB == 128 ? 2 : 8) gemm_maxplus_kernel(const MpArgs p) {
  using G = Cfg<P16, TB>;
  constexpr int NT = G::NT, BK = G::BK, BW = G::BW, UNITS = G::UNITS;
  __shared__ __align__(16) uint32_t smem[2 * G::STAGE_WORDS];

  const int tiles_n = (p.N + TB - 1) / TB, tiles_m = (p.M + TB - 1) / TB;
  const int64_t bg = blockIdx.x / (tiles_n * tiles_m);
  const int tile = (int)(blockIdx.x - bg * (tiles_n * tiles_m));
  const int64_t b = bg / p.G, g = bg - b * p.G;
  const int m0 = (tile / tiles_n) * TB, n0 = (tile % tiles_n) * TB;
  const int32_t *A = p.A + b * p.sA + g * (int64_t)p.M * p.K;
  const int32_t *B = p.B + b * p.sB + g * (int64_t)p.K * p.N;
  int32_t *C = p.C + b * p.sC + g * (int64_t)p.M * p.N;

  // a warp covers 8 tx x 4 ty: its A reads touch 4 distinct 16-byte granules (broadcast), its B reads 8 adjacent ones
  constexpr int WX = TB / 64;
  const int t = threadIdx.x, w = t >> 5, lane = t & 31;
  const int tx = (w % WX) * 8 + (lane & 7), ty = (w / WX) * 4 + (lane >> 3);          // 0 .. TB/8-1 each
  // rows: h*TB/2 + ty*4 + i.  columns, 16-bit form: tx*8 + 2j + half (4 packed words); 32-bit form: h*TB/2 + tx*4 + j
  constexpr int NACC = P16 ? 4 : 8;
  uint32_t acc[8][NACC];
#pragma unroll
  for (int i = 0; i < 8; i++)
#pragma unroll
    for (int j = 0; j < NACC; j++) acc[i][j] = P16 ? 0u : (uint32_t)NEG_INF;

  int32_t ra[UNITS][4], rb[UNITS][4];                            // the next chunk on its way global -> shared memory
  auto load = [&](int c) {
    const int k0 = c * BK;
#pragma unroll
    for (int u = 0; u < UNITS; u++) {
      const int idx = t + u * NT;
      int gm, gk;                                                // first element of the unit; its 4 run along k (row-major) or m
      if (A_KMAJOR) { gk = k0 + idx / (TB / 4); gm = m0 + 4 * (idx % (TB / 4)); }
      else { gm = m0 + idx / (BK / 4); gk = k0 + 4 * (idx % (BK / 4)); }
      const int64_t gi = A_KMAJOR ? (int64_t)gk * p.M + gm : (int64_t)gm * p.K + gk;
      const bool in4 = A_KMAJOR ? (gk < p.K && gm + 4 <= p.M) : (gm < p.M && gk + 4 <= p.K);
      if (p.vecA && in4) {
        const int4 v = __ldg(reinterpret_cast<const int4 *>(A + gi));
        ra[u][0] = v.x; ra[u][1] = v.y; ra[u][2] = v.z; ra[u][3] = v.w;
      } else {
#pragma unroll
        for (int j = 0; j < 4; j++) {
          const bool in = A_KMAJOR ? (gk < p.K && gm + j < p.M) : (gm < p.M && gk + j < p.K);
          ra[u][j] = in ? __ldg(A + gi + j) : NEG_INF;
        }
      }
    }
#pragma unroll
    for (int u = 0; u < UNITS; u++) {
      const int idx = t + u * NT;
      const int gk = k0 + idx / (TB / 4), gn = n0 + 4 * (idx % (TB / 4));
      const int64_t gi = (int64_t)gk * p.N + gn;
      if (p.vecB && gk < p.K && gn + 4 <= p.N) {
        const int4 v = __ldg(reinterpret_cast<const int4 *>(B + gi));
        rb[u][0] = v.x; rb[u][1] = v.y; rb[u][2] = v.z; rb[u][3] = v.w;
      } else {
#pragma unroll
        for (int j = 0; j < 4; j++) rb[u][j] = (gk < p.K && gn + j < p.N) ? __ldg(B + gi + j) : NEG_INF;
      }
    }
  };
  // interior tile with 16-byte access: element offsets of this thread's units are fixed, only the chunk base moves
  const bool interior = p.vecA && p.vecB && m0 + TB <= p.M && n0 + TB <= p.N &&
                        (int64_t)p.M * p.K < (1ll << 31) && (int64_t)p.K * p.N < (1ll << 31);      // 32-bit element offsets
  int offA[UNITS], offB[UNITS];
#pragma unroll
  for (int u = 0; u < UNITS; u++) {
    const int idx = t + u * NT;
    offA[u] = A_KMAJOR ? (idx / (TB / 4)) * p.M + m0 + 4 * (idx % (TB / 4)) : (m0 + idx / (BK / 4)) * p.K + 4 * (idx % (BK / 4));
    offB[u] = (idx / (TB / 4)) * p.N + n0 + 4 * (idx % (TB / 4));
  }
  auto load_fast = [&](int c) {
    const int32_t *Ac = A + (A_KMAJOR ? (int64_t)c * BK * p.M : (int64_t)c * BK);
    const int32_t *Bc = B + (int64_t)c * BK * p.N;
#pragma unroll
    for (int u = 0; u < UNITS; u++) {
      const int4 v = __ldg(reinterpret_cast<const int4 *>(Ac + offA[u]));
      ra[u][0] = v.x; ra[u][1] = v.y; ra[u][2] = v.z; ra[u][3] = v.w;
    }
#pragma unroll
    for (int u = 0; u < UNITS; u++) {
      const int4 v = __ldg(reinterpret_cast<const int4 *>(Bc + offB[u]));
      rb[u][0] = v.x; rb[u][1] = v.y; rb[u][2] = v.z; rb[u][3] = v.w;
    }
  };
  auto store = [&](int buf) {
    uint32_t *sA = smem + buf * G::STAGE_WORDS, *sB = sA + BK * TB;
#pragma unroll
    for (int u = 0; u < UNITS; u++) {
      const int idx = t + u * NT;
      if (A_KMAJOR) {
        const int kk = idx / (TB / 4), q = idx % (TB / 4);
        *reinterpret_cast<uint4 *>(sA + kk * TB + 4 * q) =
            make_uint4(enc_a<P16>(ra[u][0]), enc_a<P16>(ra[u][1]), enc_a<P16>(ra[u][2]), enc_a<P16>(ra[u][3]));
      } else {
        const int r = idx / (BK / 4), kq = idx % (BK / 4);
        const int rs = r ^ (kq * G::SWZ);                         // a warp's 32 stores of one j fall into 32 distinct banks
#pragma unroll
        for (int j = 0; j < 4; j++) sA[(4 * kq + j) * TB + rs] = enc_a<P16>(ra[u][j]);
      }
    }
#pragma unroll
    for (int u = 0; u < UNITS; u++) {
      const int idx = t + u * NT;
      const int kk = idx / (TB / 4), q = idx % (TB / 4);
      if (P16)
        *reinterpret_cast<uint2 *>(sB + kk * BW + 2 * q) =
            make_uint2(pack2(rb[u][0], rb[u][1]), pack2(rb[u][2], rb[u][3]));
      else
        *reinterpret_cast<uint4 *>(sB + kk * BW + 4 * q) =
            make_uint4(canon32(rb[u][0]), canon32(rb[u][1]), canon32(rb[u][2]), canon32(rb[u][3]));
    }
  };
  auto compute = [&](int buf) {
    const uint32_t *sA = smem + buf * G::STAGE_WORDS, *sB = sA + BK * TB;
#pragma unroll
    for (int kk = 0; kk < BK; kk++) {
      const int sw = A_KMAJOR ? 0 : (kk >> 2) * G::SWZ;          // undo the store swizzle (a multiple of 4: the 16 bytes stay together)
      uint32_t a[8], bv[NACC];
      lds4(sA + kk * TB + ((ty * 4) ^ sw), a);
      lds4(sA + kk * TB + ((TB / 2 + ty * 4) ^ sw), a + 4);
      if (P16) lds4(sB + kk * BW + tx * 4, bv);
      else { lds4(sB + kk * BW + tx * 4, bv); lds4(sB + kk * BW + TB / 2 + tx * 4, bv + 4); }
#pragma unroll
      for (int i = 0; i < 8; i++)
#pragma unroll
        for (int j = 0; j < NACC; j++)
          acc[i][j] = P16 ? __viaddmax_s16x2(a[i], bv[j], acc[i][j])
                          : (uint32_t)__viaddmax_s32((int32_t)a[i], (int32_t)bv[j], (int32_t)acc[i][j]);
    }
  };

  const int n_chunks = (p.K + BK - 1) / BK;
  const int n_fast = interior ? p.K / BK : 0;                    // chunks 0 .. n_fast-1 need no bounds checks
  if (n_fast > 0) load_fast(0); else load(0);
  store(0);
  __syncthreads();
  for (int c = 0; c < n_chunks; c++) {
    const bool more = c + 1 < n_chunks;
    if (c + 1 < n_fast) load_fast(c + 1);
    else if (more) load(c + 1);
    compute(c & 1);
    if (more) store((c + 1) & 1);        // the other buffer: last read in compute(c - 1), before the barrier that ended it
    __syncthreads();
  }

  // ---------------- epilogue: decode, canonicalise, store ----------------
#pragma unroll
  for (int i = 0; i < 8; i++) {
    const int gm = m0 + (i >> 2) * (TB / 2) + ty * 4 + (i & 3);
    if (gm >= p.M) continue;
#pragma unroll
    for (int q = 0; q < 2; q++) {                                // four consecutive columns at a time
      const int gn = n0 + (P16 ? tx * 8 + 4 * q : q * (TB / 2) + tx * 4);
      int32_t e[4];
#pragma unroll
      for (int j = 0; j < 4; j++) {
        if (P16) {
          const uint32_t hv = (acc[i][2 * q + (j >> 1)] >> ((j & 1) * 16)) & 0xffffu;
          e[j] = hv >= (uint32_t)FINITE2 ? (int32_t)hv - 2 * BIAS : NEG_INF;
        } else {
          const int32_t v = (int32_t)acc[i][q * 4 + j];
          e[j] = v < ZERO_BELOW ? NEG_INF : v;
        }
      }
      const int64_t o = (int64_t)gm * p.N + gn;
      if (p.vecC && gn + 4 <= p.N) *reinterpret_cast<int4 *>(C + o) = make_int4(e[0], e[1], e[2], e[3]);
      else {
#pragma unroll
        for (int j = 0; j < 4; j++) if (gn + j < p.N) C[o + j] = e[j];
      }
    }
  }
}

inline bool al16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

template <bool KM, bool P16, int TB>
void launch_mp(const MpArgs &a, int64_t batch, cudaStream_t st) {
  const int64_t n_cta = (int64_t)((a.N + TB - 1) / TB) * ((a.M + TB - 1) / TB) * batch * a.G;
  gemm_maxplus_kernel<KM, P16, TB><<<dim3((unsigned)n_cta), Cfg<P16, TB>::NT, 0, st>>>(a);
}

}  // namespace

// C = A (x) B over max-plus on the energy planes.  energy_bits <= 11 (every finite |energy| < 2^11, the zero element
// exactly NEG_INF) selects the packed 16-bit form, anything else the 32-bit form.
void launch_gemm_maxplus(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor, const int32_t *A, const int32_t *B,
                         int32_t *C, int64_t sA, int64_t sB, int64_t sC, int energy_bits, cudaStream_t st) {
  MpArgs a{G, M, N, K, A, B, C, sA, sB, sC, 0, 0, 0};
  const int ldA = a_kmajor ? M : K;
  a.vecA = (ldA % 4 == 0) && (sA % 4 == 0) && (((int64_t)M * K) % 4 == 0 || G == 1) && al16(A);
  a.vecB = (N % 4 == 0) && (sB % 4 == 0) && (((int64_t)K * N) % 4 == 0 || G == 1) && al16(B);
  a.vecC = (N % 4 == 0) && (sC % 4 == 0) && (((int64_t)M * N) % 4 == 0 || G == 1) && al16(C);
  // the 64 x 64 tile: where a 128-row tile would be >= 75 % padding, and where there are fewer 128 x 128 tiles than SMs
  const int64_t n_cta128 = (int64_t)((M + 127) / 128) * ((N + 127) / 128) * batch * G;
  const bool small = (M <= 64 && N <= 64) || n_cta128 < 148;
  const bool p16 = energy_bits <= 11;
#define BBTN_MP(KM, P, T) launch_mp<KM, P, T>(a, batch, st)
  if (a_kmajor) {
    if (p16) { if (small) BBTN_MP(true, true, 64); else BBTN_MP(true, true, 128); }
    else { if (small) BBTN_MP(true, false, 64); else BBTN_MP(true, false, 128); }
  } else {
    if (p16) { if (small) BBTN_MP(false, true, 64); else BBTN_MP(false, true, 128); }
    else { if (small) BBTN_MP(false, false, 64); else BBTN_MP(false, false, 128); }
  }
#undef BBTN_MP
}

}  // namespace bbtn
