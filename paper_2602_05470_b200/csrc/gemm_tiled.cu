// gemm_tiled.cu -- K3 v2: batched counting-tropical GEMM on the integer CUDA cores of sm_100a.
//
//   C[b,g,m,n] = (+)_k A[b,g,m,k] (.) B[b,g,k,n]          (PAPER.md:51 Eq. 2 evaluated pairwise, :57)
//   (ea,ca) (.) (eb,cb) = (ea+eb, ca*cb);  (+) keeps the max energy, adds counts on ties.
//
// Tensor cores cannot evaluate max-plus (north_star), so the design goal is the smallest number of
// integer-pipe instructions per tropical FMA.  The reduction over k is done chunk by chunk (BK terms),
// two passes per chunk over the same shared-memory tile:
//   pass 1  E <- max(E, ea+eb)                 one fused add-max (VIADDMNMX, ALU pipe) per FMA
//   reset   where E changed, the count of the old maximum is dropped (2 instructions per BK FMAs)
//   pass 2  if (ea+eb == E) c += ca*cb          add + compare + predicated multiply-add per FMA
// = 4 instructions per FMA, two on the ALU pipe and two that can run on the FMA pipe (IMAD), against
// ~16 for a literal transcription of (+)/(.).  Pass 2 only ever compares against the final maximum
// of everything seen so far, so the result is exactly the definition (bit-exact, order-free).
//
// CTA tile 128x128, 256 threads, 8x8 outputs per thread (2x2 blocks of 4x4 so that every operand
// fetch is one LDS.128), BK = 16, three cp.async stages, one barrier per chunk.  Operands stay in
// their global layout in shared memory (row-major A is consumed four k at a time), so interior tiles
// move with 16-byte cp.async only; ragged or unaligned tiles take a guarded scalar fill that writes
// the zero element (-inf, 0) outside the matrix.
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

constexpr int BM = 128, BN = 128, BK = 16, NT = 256, STAGES = 3;
constexpr int AE_LD = BK + 4;            // row-major A energies: [BM][AE_LD] int32 (row stride 80 B)
constexpr int AC_LD = BK + 2;            // row-major A counts:   [BM][AC_LD] uint64 (row stride 144 B)
constexpr int AE_BYTES = BM * AE_LD * 4; // k-major A needs BK*BM*4 <= this
constexpr int AC_BYTES = BM * AC_LD * 8;
constexpr int BE_BYTES = BK * BN * 4;
constexpr int BC_BYTES = BK * BN * 8;
constexpr int STAGE_BYTES = AE_BYTES + AC_BYTES + BE_BYTES + BC_BYTES;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES;

enum Mode : int { ACC32 = 0, ACC64N = 1, WIDE = 2 };
// ACC32 : operand counts < 2^16 and K * max product < 2^32: 32-bit accumulators, one IMAD per FMA
// ACC64N: operand counts < 2^32: 64-bit accumulators, one IMAD.WIDE per FMA
// WIDE  : full 64x64->64 multiply-add (IMAD.WIDE + 2 IMAD)

template <int MODE> struct AccT { using T = uint64_t; };
template <> struct AccT<ACC32> { using T = uint32_t; };

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// 16-byte granule g (two counts) of a B-count row is stored at g ^ ((g >> 3) & 1): the eight lanes of a
// quarter warp read granules 2*tx (+1), which would otherwise collide pairwise on the banks.
__device__ __forceinline__ int bc_swz(int g) { return g ^ ((g >> 3) & 1); }

// pass 2 of one FMA: if (ea + eb == E) c += ca * cb
template <int MODE>
__device__ __forceinline__ void tie_fma(typename AccT<MODE>::T &c, int32_t ea, int32_t eb, int32_t E, uint64_t ca, uint64_t cb) {
  if (MODE == ACC32) {
    uint32_t c32 = (uint32_t)c;
    asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\tadd.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\t@p mad.lo.u32 %0, %4, %5, %0;\n\t}"
        : "+r"(c32) : "r"(ea), "r"(eb), "r"(E), "r"((uint32_t)ca), "r"((uint32_t)cb));
    c = c32;
  } else if (MODE == ACC64N) {
    uint64_t c64 = c;
    asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\tadd.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\t@p mad.wide.u32 %0, %4, %5, %0;\n\t}"
        : "+l"(c64) : "r"(ea), "r"(eb), "r"(E), "r"((uint32_t)ca), "r"((uint32_t)cb));
    c = c64;
  } else {
    uint64_t c64 = c;
    asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\tadd.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\t@p mad.lo.u64 %0, %4, %5, %0;\n\t}"
        : "+l"(c64) : "r"(ea), "r"(eb), "r"(E), "l"(ca), "l"(cb));
    c = c64;
  }
}

struct GemmArgs {
  int64_t G;
  int M, N, K;
  const int32_t *Ae; const uint64_t *Ac; const int32_t *Be; const uint64_t *Bc;
  int32_t *Ce; uint64_t *Cc;
  int64_t sA, sB, sC;
  int vecA, vecB, vecC;     // 16-byte paths allowed (alignment of pointers, strides and leading dimensions)
};

template <int NCB> struct Tile {
  static constexpr int BNt = 64 * NCB;
  static constexpr int BE = BK * BNt * 4, BC = BK * BNt * 8;
  static constexpr int STAGE = AE_BYTES + AC_BYTES + BE + BC;
};

// ---- global -> shared for one chunk (k0 .. k0+BK) of one operand ------------------------------
template <bool A_KMAJOR>
__device__ __forceinline__ void fill_A(const GemmArgs &p, const int32_t *__restrict__ ae, const uint64_t *__restrict__ ac,
                                       int m0, int k0, unsigned char *sAe, unsigned char *sAc) {
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

template <int NCB>
__device__ __forceinline__ void fill_B(const GemmArgs &p, const int32_t *__restrict__ be, const uint64_t *__restrict__ bc,
                                       int n0, int k0, unsigned char *sBe, unsigned char *sBc) {
  constexpr int BNt = Tile<NCB>::BNt;
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
      cp_async16(sBc + (kk * (BNt / 2) + bc_swz(q)) * 16, bc + (int64_t)(k0 + kk) * p.N + n0 + 2 * q);
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
      sc[kk * BNt + bc_swz(n >> 1) * 2 + (n & 1)] = c;
    }
  }
}

// ---- the kernel -----------------------------------------------------------------------------
template <int MODE, bool A_KMAJOR, int NCB>
__global__ void __launch_bounds__(NT, 1) gemm_tiled2_kernel(const GemmArgs p) {
  using Acc = typename AccT<MODE>::T;
  constexpr int BNt = Tile<NCB>::BNt, STAGE = Tile<NCB>::STAGE, BEb = Tile<NCB>::BE;
  constexpr int TN = 4 * NCB;
  extern __shared__ __align__(16) unsigned char smem[];

  const int tiles_n = (p.N + BNt - 1) / BNt, tiles_m = (p.M + BM - 1) / BM;
  const int64_t bg = blockIdx.x / (tiles_n * tiles_m);
  const int tile = (int)(blockIdx.x - bg * (tiles_n * tiles_m));
  const int64_t b = bg / p.G, g = bg - b * p.G;
  const int m0 = (tile / tiles_n) * BM, n0 = (tile % tiles_n) * BNt;
  const int32_t *ae = p.Ae + b * p.sA + g * (int64_t)p.M * p.K; const uint64_t *ac = p.Ac + b * p.sA + g * (int64_t)p.M * p.K;
  const int32_t *be = p.Be + b * p.sB + g * (int64_t)p.K * p.N; const uint64_t *bc = p.Bc + b * p.sB + g * (int64_t)p.K * p.N;
  int32_t *ce = p.Ce + b * p.sC + g * (int64_t)p.M * p.N; uint64_t *cc = p.Cc + b * p.sC + g * (int64_t)p.M * p.N;

  // a warp covers 8 tx x 4 ty: A fetches touch 4 distinct 16-byte granules, B fetches 8
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tx = (w & 1) * 8 + (lane & 7), ty = (w >> 1) * 4 + (lane >> 3);
  const int sw = (tx >> 2) & 1;                       // granule swizzle of the B counts
  const int bc_off0 = (2 * tx + sw) * 16, bc_off1 = (2 * tx + 1 - sw) * 16;

  int32_t E[8][TN]; Acc C[8][TN];
#pragma unroll
  for (int i = 0; i < 8; i++)
#pragma unroll
    for (int j = 0; j < TN; j++) { E[i][j] = NEG_INF; C[i][j] = 0; }

  const int n_chunks = (p.K + BK - 1) / BK;
  auto stage_ptr = [&](int c) { return smem + (c % STAGES) * STAGE; };
  auto issue = [&](int c) {
    if (c < n_chunks) {
      unsigned char *s = stage_ptr(c);
      fill_A<A_KMAJOR>(p, ae, ac, m0, c * BK, s, s + AE_BYTES);
      fill_B<NCB>(p, be, bc, n0, c * BK, s + AE_BYTES + AC_BYTES, s + AE_BYTES + AC_BYTES + BEb);
    }
    cp_async_commit();
  };
#pragma unroll
  for (int c = 0; c < STAGES - 1; c++) issue(c);

  for (int c = 0; c < n_chunks; c++) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    issue(c + STAGES - 1);
    const unsigned char *s = stage_ptr(c);
    const int32_t *sAe = reinterpret_cast<const int32_t *>(s);
    const uint64_t *sAc = reinterpret_cast<const uint64_t *>(s + AE_BYTES);
    const int32_t *sBe = reinterpret_cast<const int32_t *>(s + AE_BYTES + AC_BYTES);
    const unsigned char *sBc = s + AE_BYTES + AC_BYTES + BEb;

#pragma unroll
    for (int rb = 0; rb < 2; rb++) {
      const int mrow = rb * 64 + ty * 4;
      // ---------------- pass 1: E <- max(E, ea + eb) ----------------
      int32_t old[4][TN];
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) old[i][j] = E[rb * 4 + i][j];
#pragma unroll 1
      for (int k4 = 0; k4 < BK / 4; k4++) {
        int32_t a[4][4];                               // [kk][i]
        if (A_KMAJOR) {
#pragma unroll
          for (int kk = 0; kk < 4; kk++) {
            const int4 v = *reinterpret_cast<const int4 *>(sAe + (k4 * 4 + kk) * BM + mrow);
            a[kk][0] = v.x; a[kk][1] = v.y; a[kk][2] = v.z; a[kk][3] = v.w;
          }
        } else {
#pragma unroll
          for (int i = 0; i < 4; i++) {
            const int4 v = *reinterpret_cast<const int4 *>(sAe + (mrow + i) * AE_LD + k4 * 4);
            a[0][i] = v.x; a[1][i] = v.y; a[2][i] = v.z; a[3][i] = v.w;
          }
        }
#pragma unroll
        for (int kk = 0; kk < 4; kk++) {
          int32_t bv[TN];
#pragma unroll
          for (int cb = 0; cb < NCB; cb++) {
            const int4 v = *reinterpret_cast<const int4 *>(sBe + (k4 * 4 + kk) * BNt + cb * 64 + tx * 4);
            bv[cb * 4 + 0] = v.x; bv[cb * 4 + 1] = v.y; bv[cb * 4 + 2] = v.z; bv[cb * 4 + 3] = v.w;
          }
#pragma unroll
          for (int i = 0; i < 4; i++)
#pragma unroll
            for (int j = 0; j < TN; j++) E[rb * 4 + i][j] = __viaddmax_s32(a[kk][i], bv[j], E[rb * 4 + i][j]);
        }
      }
      // ---------------- reset: a new maximum drops the count of the old one ----------------
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < TN; j++)
          if (E[rb * 4 + i][j] != old[i][j]) C[rb * 4 + i][j] = 0;
      // ---------------- pass 2: ties add their count products ----------------
#pragma unroll 1
      for (int k4 = 0; k4 < BK / 4; k4++) {
        int32_t a[4][4]; uint64_t ca[4][4];            // [kk][i]
        if (A_KMAJOR) {
#pragma unroll
          for (int kk = 0; kk < 4; kk++) {
            const int4 v = *reinterpret_cast<const int4 *>(sAe + (k4 * 4 + kk) * BM + mrow);
            a[kk][0] = v.x; a[kk][1] = v.y; a[kk][2] = v.z; a[kk][3] = v.w;
            const ulonglong2 c0 = *reinterpret_cast<const ulonglong2 *>(sAc + (k4 * 4 + kk) * BM + mrow);
            const ulonglong2 c1 = *reinterpret_cast<const ulonglong2 *>(sAc + (k4 * 4 + kk) * BM + mrow + 2);
            ca[kk][0] = c0.x; ca[kk][1] = c0.y; ca[kk][2] = c1.x; ca[kk][3] = c1.y;
          }
        } else {
#pragma unroll
          for (int i = 0; i < 4; i++) {
            const int4 v = *reinterpret_cast<const int4 *>(sAe + (mrow + i) * AE_LD + k4 * 4);
            a[0][i] = v.x; a[1][i] = v.y; a[2][i] = v.z; a[3][i] = v.w;
            const ulonglong2 c0 = *reinterpret_cast<const ulonglong2 *>(sAc + (mrow + i) * AC_LD + k4 * 4);
            const ulonglong2 c1 = *reinterpret_cast<const ulonglong2 *>(sAc + (mrow + i) * AC_LD + k4 * 4 + 2);
            ca[0][i] = c0.x; ca[1][i] = c0.y; ca[2][i] = c1.x; ca[3][i] = c1.y;
          }
        }
#pragma unroll
        for (int kk = 0; kk < 4; kk++) {
          int32_t bv[TN]; uint64_t cbv[TN];
#pragma unroll
          for (int cb = 0; cb < NCB; cb++) {
            const int4 v = *reinterpret_cast<const int4 *>(sBe + (k4 * 4 + kk) * BNt + cb * 64 + tx * 4);
            bv[cb * 4 + 0] = v.x; bv[cb * 4 + 1] = v.y; bv[cb * 4 + 2] = v.z; bv[cb * 4 + 3] = v.w;
            const unsigned char *row = sBc + ((k4 * 4 + kk) * (BNt / 2) + cb * 32) * 16;
            const ulonglong2 c0 = *reinterpret_cast<const ulonglong2 *>(row + bc_off0);
            const ulonglong2 c1 = *reinterpret_cast<const ulonglong2 *>(row + bc_off1);
            cbv[cb * 4 + 0] = c0.x; cbv[cb * 4 + 1] = c0.y; cbv[cb * 4 + 2] = c1.x; cbv[cb * 4 + 3] = c1.y;
          }
#pragma unroll
          for (int i = 0; i < 4; i++)
#pragma unroll
            for (int j = 0; j < TN; j++)
              tie_fma<MODE>(C[rb * 4 + i][j], a[kk][i], bv[j], E[rb * 4 + i][j], ca[kk][i], cbv[j]);
        }
      }
    }
  }
  cp_async_wait<0>();

  // ---------------- epilogue: canonicalise, store ----------------
#pragma unroll
  for (int i = 0; i < 8; i++) {
    const int gm = m0 + (i >> 2) * 64 + ty * 4 + (i & 3);
    if (gm >= p.M) continue;
#pragma unroll
    for (int cb = 0; cb < NCB; cb++) {
      const int gn = n0 + cb * 64 + tx * 4;
      int32_t e[4]; uint64_t c[4];
#pragma unroll
      for (int j = 0; j < 4; j++) {
        e[j] = E[i][cb * 4 + j]; c[j] = (uint64_t)C[i][cb * 4 + j];
        if (e[j] < ZERO_BELOW) { e[j] = NEG_INF; c[j] = 0; }
      }
      const int64_t o = (int64_t)gm * p.N + gn;
      if (p.vecC && gn + 4 <= p.N) {
        *reinterpret_cast<int4 *>(ce + o) = make_int4(e[0], e[1], e[2], e[3]);
        *reinterpret_cast<ulonglong2 *>(cc + o) = make_ulonglong2(c[0], c[1]);
        *reinterpret_cast<ulonglong2 *>(cc + o + 2) = make_ulonglong2(c[2], c[3]);
      } else {
#pragma unroll
        for (int j = 0; j < 4; j++)
          if (gn + j < p.N) { ce[o + j] = e[j]; cc[o + j] = c[j]; }
      }
    }
  }
}

template <int MODE, bool A_KMAJOR, int NCB>
void launch_one(const GemmArgs &a, int64_t batch, cudaStream_t st) {
  constexpr int BNt = Tile<NCB>::BNt;
  constexpr int smem = STAGES * Tile<NCB>::STAGE;
  static bool configured = false;                      // per instantiation; the attribute is per function
  if (!configured) {
    cudaFuncSetAttribute(gemm_tiled2_kernel<MODE, A_KMAJOR, NCB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    configured = true;
  }
  const int64_t n_cta = (int64_t)((a.N + BNt - 1) / BNt) * ((a.M + BM - 1) / BM) * batch * a.G;
  gemm_tiled2_kernel<MODE, A_KMAJOR, NCB><<<dim3((unsigned)n_cta), NT, smem, st>>>(a);
}

inline bool al16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

}  // namespace

// RING_U64 only.  count_bits is the caller's bound on log2(count+1) of both operands.
void launch_gemm_tiled_u64(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                           const int32_t *Ae, const uint64_t *Ac, const int32_t *Be, const uint64_t *Bc,
                           int32_t *Ce, uint64_t *Cc, int64_t sA, int64_t sB, int64_t sC, int count_bits, cudaStream_t st) {
  GemmArgs a{G, M, N, K, Ae, Ac, Be, Bc, Ce, Cc, sA, sB, sC, 0, 0, 0};
  const int ldA = a_kmajor ? M : K;
  a.vecA = (ldA % 4 == 0) && (sA % 4 == 0) && (((int64_t)M * K) % 4 == 0 || G == 1) && al16(Ae) && al16(Ac);
  a.vecB = (N % 4 == 0) && (sB % 4 == 0) && (((int64_t)K * N) % 4 == 0 || G == 1) && al16(Be) && al16(Bc);
  a.vecC = (N % 4 == 0) && (sC % 4 == 0) && (((int64_t)M * N) % 4 == 0 || G == 1) && al16(Ce) && al16(Cc);
  int lgK = 0;
  while (((int64_t)1 << lgK) < K) lgK++;
  const int mode = (count_bits <= 16 && 2 * count_bits + lgK <= 32) ? ACC32 : (count_bits <= 32 ? ACC64N : WIDE);
  if (mode == ACC32) {
    if (a_kmajor) launch_one<ACC32, true, 2>(a, batch, st); else launch_one<ACC32, false, 2>(a, batch, st);
  } else if (mode == ACC64N) {
    if (a_kmajor) launch_one<ACC64N, true, 1>(a, batch, st); else launch_one<ACC64N, false, 1>(a, batch, st);
  } else {
    if (a_kmajor) launch_one<WIDE, true, 1>(a, batch, st); else launch_one<WIDE, false, 1>(a, batch, st);
  }
}

}  // namespace bbtn
