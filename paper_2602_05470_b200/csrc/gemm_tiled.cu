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
// Pass 1 needs only the ALU pipe and pass 2 is FMA-pipe heavy, so pass 1 of chunk c+1 is interleaved
// (same instruction stream, independent registers) with pass 2 of chunk c: both pipes stay busy.
//
// CTA tile 128x128 (128x64 with 64-bit accumulators), 256 threads, 8x8 (8x4) outputs per thread in
// 4x4 blocks so that every operand fetch is one LDS.128, BK = 16, one barrier per chunk.  Interior
// tiles arrive by 16-byte cp.async in their global layout (raw stages); a short cooperative step
// rewrites each chunk k-major with the counts narrowed to 32 bits when the caller's count_bits
// allows (converted stages).  Ragged or unaligned tiles take a guarded scalar fill that writes the
// zero element (-inf, 0) outside the matrix.
#include "gemm_stage.cuh"
#include <type_traits>

namespace bbtn {
namespace {

using namespace stage;

enum Mode : int { ACC32 = 0, ACC64N = 1, WIDE = 2, NARROW64 = 3 };
// NARROW64: operand counts < 2^14: the ties of one chunk (BK = 16 products below 2^28) are summed in a 32-bit register
//           with ACC32's one-IMAD inner loop and added to the 64-bit accumulator once per chunk -- any K, any total
// ACC32 : operand counts < 2^16 and K * max product < 2^32: 32-bit accumulators, one IMAD per FMA
// ACC64N: operand counts < 2^32: 64-bit accumulators, one IMAD.WIDE per FMA
// WIDE  : full 64x64->64 multiply-add (IMAD.WIDE + 2 IMAD)

template <int MODE> struct AccT { using T = uint64_t; };
template <> struct AccT<ACC32> { using T = uint32_t; };

// pass 2 of one FMA: if (ea + eb == E) c += ca * cb
template <int MODE, class AccR = typename AccT<MODE>::T>
__device__ __forceinline__ void tie_fma(AccR &c, int32_t ea, int32_t eb, int32_t E, uint64_t ca, uint64_t cb) {
  if (MODE == ACC32) {
    uint32_t c32 = (uint32_t)c;
    asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\tadd.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\t@p mad.lo.u32 %0, %4, %5, %0;\n\t}"
        : "+r"(c32) : "r"(ea), "r"(eb), "r"(E), "r"((uint32_t)ca), "r"((uint32_t)cb));
    c = c32;
  } else if (MODE == ACC64N) {
    // ptxas lowers a predicated 64-bit multiply-add to multiply + 2 selects + 2 adds; selecting the 32-bit
    // multiplicand instead keeps it at SEL + IMAD.WIDE (with the 64-bit accumulate fused)
    uint64_t c64 = c;
    asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\t.reg .u32 t;\n\tadd.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\t"
        "selp.u32 t, %5, 0, p;\n\tmad.wide.u32 %0, %4, t, %0;\n\t}"
        : "+l"(c64) : "r"(ea), "r"(eb), "r"(E), "r"((uint32_t)ca), "r"((uint32_t)cb));
    c = c64;
  } else {
    // full 64x64->64: low product through SEL + IMAD.WIDE, the two cross terms as predicated 32-bit IMADs
    uint64_t c64 = c;
    asm("{\n\t.reg .pred p;\n\t.reg .s32 s;\n\t.reg .u32 alo, ahi, blo, bhi, t, clo, chi;\n\t"
        "mov.b64 {alo, ahi}, %4;\n\tmov.b64 {blo, bhi}, %5;\n\t"
        "add.s32 s, %1, %2;\n\tsetp.eq.s32 p, s, %3;\n\tselp.u32 t, blo, 0, p;\n\t"
        "mad.wide.u32 %0, alo, t, %0;\n\tmov.b64 {clo, chi}, %0;\n\t"
        "@p mad.lo.u32 chi, alo, bhi, chi;\n\t@p mad.lo.u32 chi, ahi, blo, chi;\n\t"
        "mov.b64 %0, {clo, chi};\n\t}"
        : "+l"(c64) : "r"(ea), "r"(eb), "r"(E), "l"(ca), "l"(cb));
    c = c64;
  }
}

// shared memory: RAW_STAGES raw stages (cp.async targets, operands in their global layout, uint64 counts)
// followed by CONV_STAGES converted stages (k-major, counts narrowed to CT) that the FMA loops read.
template <int NCB, class CT> struct Tile {
  static constexpr int BNt = 64 * NCB;
  static constexpr int BE = BK * BNt * 4, BC = BK * BNt * 8;
  static constexpr int RAW = AE_BYTES + AC_BYTES + BE + BC;
  static constexpr int CAE = BK * BM * 4, CAC = BK * BM * (int)sizeof(CT), CBE = BK * BNt * 4, CBC = BK * BNt * (int)sizeof(CT);
  static constexpr int CONV = CAE + CAC + CBE + CBC;
  static constexpr int SMEM = RAW_STAGES * RAW + CONV_STAGES * CONV;
};

// ---- raw stage -> converted stage (k-major, counts narrowed to CT) ---------------------------
template <class CT> __device__ __forceinline__ void store_pair(CT *dst, uint64_t x, uint64_t y);
template <> __device__ __forceinline__ void store_pair<uint32_t>(uint32_t *dst, uint64_t x, uint64_t y) {
  *reinterpret_cast<uint2 *>(dst) = make_uint2((uint32_t)x, (uint32_t)y);
}
template <> __device__ __forceinline__ void store_pair<uint64_t>(uint64_t *dst, uint64_t x, uint64_t y) {
  *reinterpret_cast<ulonglong2 *>(dst) = make_ulonglong2(x, y);
}

template <bool A_KMAJOR, int NCB, class CT>
__device__ __forceinline__ void convert_stage(const unsigned char *raw, unsigned char *conv) {
  using T = Tile<NCB, CT>;
  constexpr int BNt = T::BNt;
  const int t = threadIdx.x;
  const unsigned char *rAe = raw, *rAc = raw + AE_BYTES, *rBe = raw + AE_BYTES + AC_BYTES, *rBc = rBe + T::BE;
  int32_t *cAe = reinterpret_cast<int32_t *>(conv);
  CT *cAc = reinterpret_cast<CT *>(conv + T::CAE);
  int32_t *cBe = reinterpret_cast<int32_t *>(conv + T::CAE + T::CAC);
  CT *cBc = reinterpret_cast<CT *>(conv + T::CAE + T::CAC + T::CBE);
  if (A_KMAJOR) {
#pragma unroll
    for (int idx = t; idx < BK * BM / 4; idx += NT)
      *reinterpret_cast<int4 *>(cAe + 4 * idx) = *reinterpret_cast<const int4 *>(rAe + 16 * idx);
#pragma unroll
    for (int idx = t; idx < BK * BM / 2; idx += NT) {
      const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(rAc + 16 * idx);
      store_pair<CT>(cAc + 2 * idx, v.x, v.y);
    }
  } else {
    // transpose: lane = row, so the k-major stores of a warp are contiguous; raw row strides (80 B, 144 B)
    // keep the 16-byte reads of a quarter warp on distinct banks
    const int r = t % BM, kb = (t / BM) * (BK / 2);
#pragma unroll
    for (int q = 0; q < BK / 8; q++) {
      const int4 v = *reinterpret_cast<const int4 *>(rAe + (r * AE_LD + kb + 4 * q) * 4);
      cAe[(kb + 4 * q + 0) * BM + r] = v.x; cAe[(kb + 4 * q + 1) * BM + r] = v.y;
      cAe[(kb + 4 * q + 2) * BM + r] = v.z; cAe[(kb + 4 * q + 3) * BM + r] = v.w;
    }
#pragma unroll
    for (int q = 0; q < BK / 4; q++) {
      const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(rAc + (r * AC_LD + kb + 2 * q) * 8);
      cAc[(kb + 2 * q + 0) * BM + r] = (CT)v.x; cAc[(kb + 2 * q + 1) * BM + r] = (CT)v.y;
    }
  }
#pragma unroll
  for (int idx = t; idx < BK * BNt / 4; idx += NT)
    *reinterpret_cast<int4 *>(cBe + 4 * idx) = *reinterpret_cast<const int4 *>(rBe + 16 * idx);
#pragma unroll
  for (int idx = t; idx < BK * BNt / 2; idx += NT) {
    const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(rBc + 16 * idx);
    store_pair<CT>(cBc + 2 * idx, v.x, v.y);
  }
}

__device__ __forceinline__ void load4(const uint32_t *src, uint64_t *dst) {
  const uint4 v = *reinterpret_cast<const uint4 *>(src);
  dst[0] = v.x; dst[1] = v.y; dst[2] = v.z; dst[3] = v.w;
}
__device__ __forceinline__ void load4(const uint64_t *src, uint64_t *dst) {
  const ulonglong2 v0 = *reinterpret_cast<const ulonglong2 *>(src), v1 = *reinterpret_cast<const ulonglong2 *>(src + 2);
  dst[0] = v0.x; dst[1] = v0.y; dst[2] = v1.x; dst[3] = v1.y;
}
__device__ __forceinline__ void load4(const int32_t *src, int32_t *dst) {
  const int4 v = *reinterpret_cast<const int4 *>(src);
  dst[0] = v.x; dst[1] = v.y; dst[2] = v.z; dst[3] = v.w;
}

// ---- the kernel -----------------------------------------------------------------------------
template <int MODE, bool A_KMAJOR, int NCB>
__global__ void __launch_bounds__(NT, 1) gemm_tiled3_kernel(const GemmArgs p) {
  using Acc = typename AccT<MODE>::T;
  using CT = typename std::conditional<MODE == WIDE, uint64_t, uint32_t>::type;
  using T = Tile<NCB, CT>;
  constexpr int BNt = T::BNt, TN = 4 * NCB;
  extern __shared__ __align__(16) unsigned char smem[];
  unsigned char *conv_base = smem + RAW_STAGES * T::RAW;

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

  int32_t E[8][TN]; Acc C[8][TN];
#pragma unroll
  for (int i = 0; i < 8; i++)
#pragma unroll
    for (int j = 0; j < TN; j++) { E[i][j] = NEG_INF; C[i][j] = 0; }

  const int n_chunks = (p.K + BK - 1) / BK;
  auto issue = [&](int c) {                          // global -> raw stage c % RAW_STAGES
    if (c < n_chunks) {
      unsigned char *s = smem + (c % RAW_STAGES) * T::RAW;
      fill_A<A_KMAJOR>(p, ae, ac, m0, c * BK, s, s + AE_BYTES);
      fill_B<BNt>(p, be, bc, n0, c * BK, s + AE_BYTES + AC_BYTES, s + AE_BYTES + AC_BYTES + T::BE);
    }
    cp_async_commit();
  };
  auto convert = [&](int c) {                        // raw stage -> converted stage c % CONV_STAGES
    if (c < n_chunks)
      convert_stage<A_KMAJOR, NCB, CT>(smem + (c % RAW_STAGES) * T::RAW, conv_base + (c % CONV_STAGES) * T::CONV);
  };

  // one unit: pass 2 of chunk `c` on row block rb, interleaved with pass 1 of chunk c+1 on the same rows
  auto unit = [&](auto do_p1, auto rb_tag, int c) {
    constexpr bool P1 = decltype(do_p1)::value;
    constexpr int rb = decltype(rb_tag)::value;
    const unsigned char *s2 = conv_base + (c % CONV_STAGES) * T::CONV;
    const unsigned char *s1 = conv_base + ((c + 1) % CONV_STAGES) * T::CONV;
    const int mrow = rb * 64 + ty * 4;
    const int32_t *a2e = reinterpret_cast<const int32_t *>(s2) + mrow;
    const CT *a2c = reinterpret_cast<const CT *>(s2 + T::CAE) + mrow;
    const int32_t *b2e = reinterpret_cast<const int32_t *>(s2 + T::CAE + T::CAC) + tx * 4;
    const CT *b2c = reinterpret_cast<const CT *>(s2 + T::CAE + T::CAC + T::CBE) + tx * 4;
    const int32_t *a1e = reinterpret_cast<const int32_t *>(s1) + mrow;
    const int32_t *b1e = reinterpret_cast<const int32_t *>(s1 + T::CAE + T::CAC) + tx * 4;
    int32_t En[4][TN];
    if (P1) {
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) En[i][j] = E[rb * 4 + i][j];
    }
    uint32_t c32[MODE == NARROW64 ? 4 : 1][MODE == NARROW64 ? TN : 1];       // NARROW64: this chunk's tie counts
    if (MODE == NARROW64) {
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) c32[MODE == NARROW64 ? i : 0][MODE == NARROW64 ? j : 0] = 0u;
    }
#pragma unroll 4
    for (int kk = 0; kk < BK; kk++) {
      int32_t a2[4], b2[TN]; uint64_t ca[4], cb[TN];
      load4(a2e + kk * BM, a2); load4(a2c + kk * BM, ca);
#pragma unroll
      for (int q = 0; q < NCB; q++) { load4(b2e + kk * BNt + q * 64, b2 + 4 * q); load4(b2c + kk * BNt + q * 64, cb + 4 * q); }
      int32_t a1[4], b1[TN];
      if (P1) {
        load4(a1e + kk * BM, a1);
#pragma unroll
        for (int q = 0; q < NCB; q++) load4(b1e + kk * BNt + q * 64, b1 + 4 * q);
      }
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) {
          if (P1) En[i][j] = __viaddmax_s32(a1[i], b1[j], En[i][j]);
          if (MODE == NARROW64) tie_fma<ACC32>(c32[MODE == NARROW64 ? i : 0][MODE == NARROW64 ? j : 0], a2[i], b2[j], E[rb * 4 + i][j], ca[i], cb[j]);
          else tie_fma<MODE>(C[rb * 4 + i][j], a2[i], b2[j], E[rb * 4 + i][j], ca[i], cb[j]);
        }
    }
    if (MODE == NARROW64) {
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) C[rb * 4 + i][j] += c32[MODE == NARROW64 ? i : 0][MODE == NARROW64 ? j : 0];
    }
    if (P1) {                                        // a new maximum drops the count of the old one
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < TN; j++) {
          if (En[i][j] != E[rb * 4 + i][j]) C[rb * 4 + i][j] = 0;
          E[rb * 4 + i][j] = En[i][j];
        }
    }
  };

  // ---- prologue: chunks 0 and 1 converted, chunk 2 in flight, pass 1 of chunk 0 done ----
  issue(0); issue(1);
  cp_async_wait<0>();
  __syncthreads();
  convert(0); convert(1);
  __syncthreads();
  issue(2);
  {
    const unsigned char *s1 = conv_base;
#pragma unroll
    for (int rb = 0; rb < 2; rb++) {
      const int32_t *a1e = reinterpret_cast<const int32_t *>(s1) + rb * 64 + ty * 4;
      const int32_t *b1e = reinterpret_cast<const int32_t *>(s1 + T::CAE + T::CAC) + tx * 4;
#pragma unroll 4
      for (int kk = 0; kk < BK; kk++) {
        int32_t a1[4], b1[TN];
        load4(a1e + kk * BM, a1);
#pragma unroll
        for (int q = 0; q < NCB; q++) load4(b1e + kk * BNt + q * 64, b1 + 4 * q);
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
          for (int j = 0; j < TN; j++) E[rb * 4 + i][j] = __viaddmax_s32(a1[i], b1[j], E[rb * 4 + i][j]);
      }
    }
  }

  for (int c = 0; c < n_chunks; c++) {
    cp_async_wait<0>();
    __syncthreads();
    convert(c + 2);
    issue(c + 3);
    if (c + 1 < n_chunks) {
      unit(std::true_type{}, std::integral_constant<int, 0>{}, c);
      unit(std::true_type{}, std::integral_constant<int, 1>{}, c);
    } else {
      unit(std::false_type{}, std::integral_constant<int, 0>{}, c);
      unit(std::false_type{}, std::integral_constant<int, 1>{}, c);
    }
  }
  cp_async_wait<0>();

  // ---------------- epilogue: canonicalise, store ----------------
#pragma unroll
  for (int i = 0; i < 8; i++) {
    const int gm = m0 + (i >> 2) * 64 + ty * 4 + (i & 3);
    if (gm >= p.M) continue;
#pragma unroll
    for (int q = 0; q < NCB; q++) {
      const int gn = n0 + q * 64 + tx * 4;
      int32_t e[4]; uint64_t c[4];
#pragma unroll
      for (int j = 0; j < 4; j++) {
        e[j] = E[i][q * 4 + j]; c[j] = (uint64_t)C[i][q * 4 + j];
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
  using CT = typename std::conditional<MODE == WIDE, uint64_t, uint32_t>::type;
  using T = Tile<NCB, CT>;
  static_assert(T::SMEM <= 227 * 1024, "shared memory budget");
  // per function AND per device, so set it on every launch (a cheap host-side call)
  cudaFuncSetAttribute(gemm_tiled3_kernel<MODE, A_KMAJOR, NCB>, cudaFuncAttributeMaxDynamicSharedMemorySize, T::SMEM);
  const int64_t n_cta = (int64_t)((a.N + T::BNt - 1) / T::BNt) * ((a.M + BM - 1) / BM) * batch * a.G;
  gemm_tiled3_kernel<MODE, A_KMAJOR, NCB><<<dim3((unsigned)n_cta), NT, T::SMEM, st>>>(a);
}

inline bool al16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

}  // namespace

// the packed form needs finite |energy| < 2^11 and operand counts below 2^32 (32-bit accumulators where
// 2 * count_bits + ceil(log2 K) <= 32, else the carry form or 64-bit accumulators: gemm_pack16.cu)
bool gemm_pack16_eligible(int K, int count_bits, int energy_bits) {
  (void)K;
  return count_bits <= 32 && energy_bits <= 11;
}

// RING_U64 only.  count_bits is the caller's bound on log2(count+1) of both operands.
void launch_gemm_tiled_u64(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                           const int32_t *Ae, const uint64_t *Ac, const int32_t *Be, const uint64_t *Bc,
                           int32_t *Ce, uint64_t *Cc, int64_t sA, int64_t sB, int64_t sC, int count_bits, int energy_bits,
                           cudaStream_t st) {
  GemmArgs a{G, M, N, K, Ae, Ac, Be, Bc, Ce, Cc, sA, sB, sC, 0, 0, 0};
  const int ldA = a_kmajor ? M : K;
  a.vecA = (ldA % 4 == 0) && (sA % 4 == 0) && (((int64_t)M * K) % 4 == 0 || G == 1) && al16(Ae) && al16(Ac);
  a.vecB = (N % 4 == 0) && (sB % 4 == 0) && (((int64_t)K * N) % 4 == 0 || G == 1) && al16(Be) && al16(Bc);
  a.vecC = (N % 4 == 0) && (sC % 4 == 0) && (((int64_t)M * N) % 4 == 0 || G == 1) && al16(Ce) && al16(Cc);
  int lgK = 0;
  while (((int64_t)1 << lgK) < K) lgK++;
  const int mode = (count_bits <= 16 && 2 * count_bits + lgK <= 32) ? ACC32
                   : (count_bits <= 14 ? NARROW64 : (count_bits <= 32 ? ACC64N : WIDE));
  // packed energies: 32-bit accumulators, the carry form (count_bits <= 13) or 64-bit accumulators (count_bits 15..32);
  // count_bits == 14 is faster in the 32-bit-energy NARROW64 form below (4.5 against 3.4 TFMA/s)
  if (mode != WIDE && energy_bits <= 11 && !(mode == NARROW64 && count_bits == 14)) {
    launch_gemm_pack16(batch, G, M, N, K, a_kmajor, Ae, Ac, Be, Bc, Ce, Cc, sA, sB, sC, count_bits, st);
  } else if (mode == ACC32) {
    // fewer 128 x 128 tiles than SMs: the 128 x 64 tile doubles the CTAs
    const int64_t n_cta128 = (int64_t)((M + 127) / 128) * ((N + 127) / 128) * batch * G;
    if (n_cta128 < 148) { if (a_kmajor) launch_one<ACC32, true, 1>(a, batch, st); else launch_one<ACC32, false, 1>(a, batch, st); }
    else if (a_kmajor) launch_one<ACC32, true, 2>(a, batch, st); else launch_one<ACC32, false, 2>(a, batch, st);
  } else if (mode == NARROW64) {
    if (a_kmajor) launch_one<NARROW64, true, 1>(a, batch, st); else launch_one<NARROW64, false, 1>(a, batch, st);
  } else if (mode == ACC64N) {
    if (a_kmajor) launch_one<ACC64N, true, 1>(a, batch, st); else launch_one<ACC64N, false, 1>(a, batch, st);
  } else {
    if (a_kmajor) launch_one<WIDE, true, 1>(a, batch, st); else launch_one<WIDE, false, 1>(a, batch, st);
  }
}

}  // namespace bbtn
