// gemm_pack16.cu -- K3, packed form: batched counting-tropical GEMM with TWO outputs per integer instruction.
//
//   C[b,g,m,n] = (+)_k A[b,g,m,k] (.) B[b,g,k,n]          (PAPER.md:51 Eq. 2 evaluated pairwise, :57)
//
// When the caller promises small energies (|e| < 2^11 for every finite operand energy; the zero element is
// exactly BBTN_NEG_INF) and small counts (32-bit accumulators suffice), the energy half of the semiring fits
// 16 bits and two neighbouring output columns share one 32-bit register:
//   pass 1  E2 <- max(E2, a2 + b2)           one VIADDMNMX.S16x2 per TWO tropical FMAs (a2 = (a, a), b2 = (b_n, b_n+1))
//   pass 2  s2 = a2 + b2;  (p, q) = (s2 == E2) per half;  @p c_n += ca*cb_n;  @q c_n+1 += ca*cb_n+1
//           = one 32-bit add + one HSETP2.EQ (two predicates from one instruction) + two predicated IMADs
// = 2.5 integer-pipe instructions per FMA against 4 for the 32-bit form of gemm_tiled.cu; the result is the same
// integers (bit-exact: the tests compare with the oracle).
//
// Encoding.  Each half holds enc(e) = e + BIAS for a finite energy and 0 for the zero element, with BIAS = 11903
// and |e| <= 3967, so that
//   * every half is a non-negative 15-bit number and the sum of two halves stays below 2^15: a plain 32-bit
//     add of two packed words never carries from the low into the high half;
//   * finite + finite >= 2 (BIAS - 3967) = 15872 > zero + finite: "the sum is finite" is "half >= 15872";
//   * every half is below 0x7C00: read as an fp16 bit pattern it is a finite non-negative number, and for
//     those the order (and equality) of bit patterns is the order of the numbers -- which is why the
//     half-precision compare HSETP2 can deliver the integer tie test for both halves at once.
// Tile 128 x 128, 512 threads (4 warps per SM sub-partition), 4 x 8 outputs per thread (4 rows x 4 packed column pairs), BK = 16, raw cp.async
// stages + converted (encoded, k-major) stages as in gemm_tiled.cu.
#include "gemm_stage.cuh"
#include <type_traits>

namespace bbtn {
namespace {

using namespace stage;

constexpr int BIAS = 11903, FINITE2 = 15872;   // enc(e) = e + BIAS;  half >= FINITE2  <=>  finite sum
// count accumulators:
//   CM_ACC32    32-bit (2 * count_bits + ceil(log2 K) <= 32)
//   CM_CARRY31  operand counts < 2^13, any K: the 32-bit accumulator is kept below 2^31 at chunk boundaries (a chunk adds
//               16 products < 2^26, so it cannot wrap inside a chunk) and its bit 31 is moved into a second 32-bit register
//               after every chunk: total = hi * 2^31 + lo < 2^63.  Inner loop = CM_ACC32's.
//   CM_WIDE64   operand counts < 2^32: 64-bit accumulators, SEL + IMAD.WIDE per FMA
enum CountMode : int { CM_ACC32 = 0, CM_CARRY31 = 1, CM_WIDE64 = 2 };
// tile TB x TB (128: the general case; 64: matrices with M, N <= 64, where the big tile would be mostly padding),
// TB*TB/32 threads: 4 x 8 outputs each
template <int TB> struct Cfg {
  static constexpr int BM = TB, BN = TB, PT = TB * TB / 32;
  static constexpr int AE_B = BM * AE_LD * 4, AC_B = BM * AC_LD * 8;            // raw A planes (row-major form is the larger one)
  static constexpr int RAW = AE_B + AC_B + BK * BN * 4 + BK * BN * 8;
  static constexpr int CAE = BK * BM * 4, CAC = BK * BM * 4, CBE = BK * (BN / 2) * 4, CBC = BK * BN * 4;
  static constexpr int CONV = CAE + CAC + CBE + CBC;
  static constexpr int SMEM = RAW_STAGES * RAW + CONV_STAGES * CONV;
  static constexpr int MIN_CTAS = TB == 128 ? 1 : 2;
  static_assert(SMEM * MIN_CTAS <= 227 * 1024, "shared memory budget");
};

__device__ __forceinline__ uint32_t enc(int32_t e) { return e < ZERO_BELOW ? 0u : (uint32_t)(e + BIAS); }

// pass 2 for one packed pair: s2 = a2 + b2; the halves that equal E2 add their count products.
// ON_ALU: the add is written with a carry-out, which only the ALU pipe's IADD3 has; left alone ptxas issues every one
// of these adds as IMAD.IADD and the FMA pipe (2 IMAD + 1 add per pair) becomes the bottleneck while the ALU pipe
// (VIADDMNMX + HSETP2) idles a third of the time.  Alternating the two forms balances the pipes.
template <bool ON_ALU>
__device__ __forceinline__ void tie2(uint32_t &c_lo, uint32_t &c_hi, uint32_t a2, uint32_t b2, uint32_t E2, uint32_t ca,
                                     uint32_t cb_lo, uint32_t cb_hi) {
  if (ON_ALU)
    asm("{\n\t.reg .pred p, q;\n\t.reg .b32 s;\n\t"
        "add.cc.u32 s, %2, %3;\n\t"
        "setp.eq.f16x2 p|q, s, %4;\n\t"
        "@p mad.lo.u32 %0, %5, %6, %0;\n\t"
        "@q mad.lo.u32 %1, %5, %7, %1;\n\t}"
        : "+r"(c_lo), "+r"(c_hi) : "r"(a2), "r"(b2), "r"(E2), "r"(ca), "r"(cb_lo), "r"(cb_hi));
  else
    asm("{\n\t.reg .pred p, q;\n\t.reg .b32 s;\n\t"
        "add.u32 s, %2, %3;\n\t"
        "setp.eq.f16x2 p|q, s, %4;\n\t"
        "@p mad.lo.u32 %0, %5, %6, %0;\n\t"
        "@q mad.lo.u32 %1, %5, %7, %1;\n\t}"
        : "+r"(c_lo), "+r"(c_hi) : "r"(a2), "r"(b2), "r"(E2), "r"(ca), "r"(cb_lo), "r"(cb_hi));
}
// the same with 64-bit accumulators and 32-bit operand counts (CM_WIDE64): ptxas turns a predicated mad.wide into
// multiply + add + add-with-carry + two selects, so the predicate selects the multiplicand instead (SEL + IMAD.WIDE)
__device__ __forceinline__ void tie2w(uint64_t &c_lo, uint64_t &c_hi, uint32_t a2, uint32_t b2, uint32_t E2, uint32_t ca,
                                      uint32_t cb_lo, uint32_t cb_hi) {
  asm("{\n\t.reg .pred p, q;\n\t.reg .b32 s, t0, t1;\n\t"
      "add.u32 s, %2, %3;\n\t"
      "setp.eq.f16x2 p|q, s, %4;\n\t"
      "selp.u32 t0, %6, 0, p;\n\t"
      "selp.u32 t1, %7, 0, q;\n\t"
      "mad.wide.u32 %0, %5, t0, %0;\n\t"
      "mad.wide.u32 %1, %5, t1, %1;\n\t}"
      : "+l"(c_lo), "+l"(c_hi) : "r"(a2), "r"(b2), "r"(E2), "r"(ca), "r"(cb_lo), "r"(cb_hi));
}
__device__ __forceinline__ void reset2w(uint64_t &c_lo, uint64_t &c_hi, uint32_t En2, uint32_t E2) {
  asm("{\n\t.reg .pred p, q;\n\t"
      "setp.ne.f16x2 p|q, %2, %3;\n\t"
      "@p mov.u64 %0, 0;\n\t"
      "@q mov.u64 %1, 0;\n\t}"
      : "+l"(c_lo), "+l"(c_hi) : "r"(En2), "r"(E2));
}
// a new maximum in a half drops the count of the old one
__device__ __forceinline__ void reset2(uint32_t &c_lo, uint32_t &c_hi, uint32_t En2, uint32_t E2) {
  asm("{\n\t.reg .pred p, q;\n\t"
      "setp.ne.f16x2 p|q, %2, %3;\n\t"
      "@p mov.u32 %0, 0;\n\t"
      "@q mov.u32 %1, 0;\n\t}"
      : "+r"(c_lo), "+r"(c_hi) : "r"(En2), "r"(E2));
}

// raw stage (operands in their global layout) -> converted stage: encoded energies, A k-major with the value in both
// halves, B as packed column pairs laid out [k][tx][q][p] (column = q*64 + tx*4 + 2p + half), counts narrowed to 32 bits
template <bool A_KMAJOR, int TB>
__device__ __forceinline__ void convert_pack16(const unsigned char *raw, unsigned char *conv) {
  using G = Cfg<TB>;
  constexpr int BM = G::BM, BN = G::BN, PT = G::PT;
  const int t = threadIdx.x;
  const unsigned char *rAe = raw, *rAc = raw + G::AE_B, *rBe = raw + G::AE_B + G::AC_B, *rBc = rBe + BK * BN * 4;
  uint32_t *cAe = reinterpret_cast<uint32_t *>(conv);
  uint32_t *cAc = reinterpret_cast<uint32_t *>(conv + G::CAE);
  uint32_t *cBe = reinterpret_cast<uint32_t *>(conv + G::CAE + G::CAC);
  uint32_t *cBc = reinterpret_cast<uint32_t *>(conv + G::CAE + G::CAC + G::CBE);
  if (A_KMAJOR) {
#pragma unroll
    for (int idx = t; idx < BK * BM / 4; idx += PT) {
      const int4 v = *reinterpret_cast<const int4 *>(rAe + 16 * idx);
      *reinterpret_cast<uint4 *>(cAe + 4 * idx) = make_uint4(enc(v.x) * 0x10001u, enc(v.y) * 0x10001u, enc(v.z) * 0x10001u, enc(v.w) * 0x10001u);
    }
#pragma unroll
    for (int idx = t; idx < BK * BM / 2; idx += PT) {
      const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(rAc + 16 * idx);
      *reinterpret_cast<uint2 *>(cAc + 2 * idx) = make_uint2((uint32_t)v.x, (uint32_t)v.y);
    }
  } else {
    // transpose: lane = row, so the k-major stores of a warp are contiguous; PT / BM thread groups share the BK values of k
    constexpr int KPER = BK / (PT / BM);                   // 4 (TB = 128) or 8 (TB = 64) k per thread
    const int r = t % BM, kb = (t / BM) * KPER;
#pragma unroll
    for (int q = 0; q < KPER / 4; q++) {
      const int4 v = *reinterpret_cast<const int4 *>(rAe + (r * AE_LD + kb + 4 * q) * 4);
      cAe[(kb + 4 * q + 0) * BM + r] = enc(v.x) * 0x10001u; cAe[(kb + 4 * q + 1) * BM + r] = enc(v.y) * 0x10001u;
      cAe[(kb + 4 * q + 2) * BM + r] = enc(v.z) * 0x10001u; cAe[(kb + 4 * q + 3) * BM + r] = enc(v.w) * 0x10001u;
    }
#pragma unroll
    for (int q = 0; q < KPER / 2; q++) {
      const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(rAc + (r * AC_LD + kb + 2 * q) * 8);
      cAc[(kb + 2 * q + 0) * BM + r] = (uint32_t)v.x; cAc[(kb + 2 * q + 1) * BM + r] = (uint32_t)v.y;
    }
  }
#pragma unroll
  for (int idx = t; idx < BK * BN / 4; idx += PT) {            // 4 consecutive columns -> two packed words
    const int kk = idx / (BN / 4), c4 = idx % (BN / 4);       // columns 4*c4 .. 4*c4+3: q = c4 / (BN/8), tx = c4 % (BN/8)
    const int4 v = *reinterpret_cast<const int4 *>(rBe + 16 * idx);
    *reinterpret_cast<uint2 *>(cBe + kk * (BN / 2) + (c4 % (BN / 8)) * 4 + (c4 / (BN / 8)) * 2) =
        make_uint2(enc(v.x) | (enc(v.y) << 16), enc(v.z) | (enc(v.w) << 16));
  }
#pragma unroll
  for (int idx = t; idx < BK * BN / 2; idx += PT) {
    const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(rBc + 16 * idx);
    *reinterpret_cast<uint2 *>(cBc + 2 * idx) = make_uint2((uint32_t)v.x, (uint32_t)v.y);
  }
}

__device__ __forceinline__ void lds4(const uint32_t *src, uint32_t *dst) {
  const uint4 v = *reinterpret_cast<const uint4 *>(src);
  dst[0] = v.x; dst[1] = v.y; dst[2] = v.z; dst[3] = v.w;
}

template <bool A_KMAJOR, int TB, int CM>
__global__ void __launch_bounds__(Cfg<TB>::PT, Cfg<TB>::MIN_CTAS) gemm_pack16_kernel(const GemmArgs p) {
  static_assert(CM == CM_ACC32 || TB == 64, "the 64-bit count modes need more than the 128 registers of the 512-thread tile");
  using G = Cfg<TB>;
  constexpr int BM = G::BM, BN = G::BN, PT = G::PT;
  constexpr int P_RAW = G::RAW, P_CONV = G::CONV, P_CAE = G::CAE, P_CAC = G::CAC, P_CBE = G::CBE;
  extern __shared__ __align__(16) unsigned char smem[];
  unsigned char *conv_base = smem + RAW_STAGES * P_RAW;

  const int tiles_n = (p.N + BN - 1) / BN, tiles_m = (p.M + BM - 1) / BM;
  const int64_t bg = blockIdx.x / (tiles_n * tiles_m);
  const int tile = (int)(blockIdx.x - bg * (tiles_n * tiles_m));
  const int64_t b = bg / p.G, g = bg - b * p.G;
  const int m0 = (tile / tiles_n) * BM, n0 = (tile % tiles_n) * BN;
  const int32_t *ae = p.Ae + b * p.sA + g * (int64_t)p.M * p.K; const uint64_t *ac = p.Ac + b * p.sA + g * (int64_t)p.M * p.K;
  const int32_t *be = p.Be + b * p.sB + g * (int64_t)p.K * p.N; const uint64_t *bc = p.Bc + b * p.sB + g * (int64_t)p.K * p.N;
  int32_t *ce = p.Ce + b * p.sC + g * (int64_t)p.M * p.N; uint64_t *cc = p.Cc + b * p.sC + g * (int64_t)p.M * p.N;

  // a warp covers 8 tx x 4 ty: A fetches touch 4 distinct 16-byte granules, B fetches 8; 16 warps = 2 (tx) x 8 (ty)
  constexpr int WX = BN / 64;                               // warps side by side along the columns (8 tx each)
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tx = (w % WX) * 8 + (lane & 7), ty = (w / WX) * 4 + (lane >> 3);      // tx 0..BN/8-1, ty 0..BM/4-1

  // rows: ty*4 + i (i = 0..3); columns: q*BN/2 + tx*4 + 2p + half (q = 0,1; p = 0,1)
  using AccC = typename std::conditional<CM == CM_WIDE64, uint64_t, uint32_t>::type;
  uint32_t E2[4][4]; AccC C[4][8];
  uint32_t H[CM == CM_CARRY31 ? 4 : 1][8];                  // CM_CARRY31: carries out of bit 31 of C
#pragma unroll
  for (int i = 0; i < 4; i++) {
#pragma unroll
    for (int j = 0; j < 4; j++) E2[i][j] = 0u;
#pragma unroll
    for (int j = 0; j < 8; j++) { C[i][j] = 0; if (CM == CM_CARRY31) H[i][j] = 0u; }
  }

  const int n_chunks = (p.K + BK - 1) / BK;
  auto issue = [&](int c) {
    if (c < n_chunks) {
      unsigned char *s = smem + (c % RAW_STAGES) * P_RAW;
      fill_A<A_KMAJOR, PT, BM>(p, ae, ac, m0, c * BK, s, s + G::AE_B);
      fill_B<BN, PT>(p, be, bc, n0, c * BK, s + G::AE_B + G::AC_B, s + G::AE_B + G::AC_B + BK * BN * 4);
    }
    cp_async_commit();
  };
  auto convert = [&](int c) {
    if (c < n_chunks) convert_pack16<A_KMAJOR, TB>(smem + (c % RAW_STAGES) * P_RAW, conv_base + (c % CONV_STAGES) * P_CONV);
  };

  // pass 1 of one chunk on row block rb: En2 <- max(En2, a2 + b2)
  auto pass1 = [&](const unsigned char *s1, uint32_t (&En)[4][4]) {
    const uint32_t *a1e = reinterpret_cast<const uint32_t *>(s1) + ty * 4;
    const uint32_t *b1e = reinterpret_cast<const uint32_t *>(s1 + P_CAE + P_CAC) + tx * 4;
#pragma unroll 4
    for (int kk = 0; kk < BK; kk++) {
      uint32_t a1[4], b1[4];
      lds4(a1e + kk * BM, a1); lds4(b1e + kk * (BN / 2), b1);
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) En[i][j] = __viaddmax_s16x2(a1[i], b1[j], En[i][j]);
    }
  };

  // one unit: pass 2 of chunk c on row block rb, interleaved with pass 1 of chunk c+1 on the same rows
  auto unit = [&](auto do_p1, int c) {
    constexpr bool P1 = decltype(do_p1)::value;
    constexpr int rb = 0;
    const unsigned char *s2 = conv_base + (c % CONV_STAGES) * P_CONV;
    const unsigned char *s1 = conv_base + ((c + 1) % CONV_STAGES) * P_CONV;
    const int mrow = ty * 4;
    const uint32_t *a2e = reinterpret_cast<const uint32_t *>(s2) + mrow;
    const uint32_t *a2c = reinterpret_cast<const uint32_t *>(s2 + P_CAE) + mrow;
    const uint32_t *b2e = reinterpret_cast<const uint32_t *>(s2 + P_CAE + P_CAC) + tx * 4;
    const uint32_t *b2c = reinterpret_cast<const uint32_t *>(s2 + P_CAE + P_CAC + P_CBE) + tx * 4;
    const uint32_t *a1e = reinterpret_cast<const uint32_t *>(s1) + mrow;
    const uint32_t *b1e = reinterpret_cast<const uint32_t *>(s1 + P_CAE + P_CAC) + tx * 4;
    uint32_t En[4][4];
    if (P1) {
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) En[i][j] = E2[rb * 4 + i][j];
    }
#pragma unroll 4
    for (int kk = 0; kk < BK; kk++) {
      uint32_t a2[4], ca[4], b2[4], cb[8];
      lds4(a2e + kk * BM, a2); lds4(a2c + kk * BM, ca);
      lds4(b2e + kk * (BN / 2), b2);
      lds4(b2c + kk * BN, cb); lds4(b2c + kk * BN + BN / 2, cb + 4);
      uint32_t a1[4], b1[4];
      if (P1) { lds4(a1e + kk * BM, a1); lds4(b1e + kk * (BN / 2), b1); }
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {                        // j = q*2 + p: columns q*64 + tx*4 + 2p, +1
          if (P1) En[i][j] = __viaddmax_s16x2(a1[i], b1[j], En[i][j]);
          if constexpr (CM == CM_WIDE64)
            tie2w(C[i][2 * j], C[i][2 * j + 1], a2[i], b2[j], E2[i][j], ca[i], cb[2 * j], cb[2 * j + 1]);
          else if ((i * 4 + j) % 8 < 5)                  // 10 of 16 adds on the ALU pipe: ALU 42 / FMA 38 instructions per kk
            tie2<true>(C[rb * 4 + i][2 * j], C[rb * 4 + i][2 * j + 1], a2[i], b2[j], E2[rb * 4 + i][j], ca[i], cb[2 * j], cb[2 * j + 1]);
          else
            tie2<false>(C[rb * 4 + i][2 * j], C[rb * 4 + i][2 * j + 1], a2[i], b2[j], E2[rb * 4 + i][j], ca[i], cb[2 * j], cb[2 * j + 1]);
        }
    }
    if constexpr (CM == CM_CARRY31) {                    // once per chunk: move bit 31 of the running sum into the carry register
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 8; j++) { H[i][j] += C[i][j] >> 31; C[i][j] &= 0x7fffffffu; }
    }
    if (P1) {
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {
          if constexpr (CM == CM_WIDE64) reset2w(C[i][2 * j], C[i][2 * j + 1], En[i][j], E2[i][j]);
          else {
            reset2(C[rb * 4 + i][2 * j], C[rb * 4 + i][2 * j + 1], En[i][j], E2[rb * 4 + i][j]);
            if constexpr (CM == CM_CARRY31) reset2(H[i][2 * j], H[i][2 * j + 1], En[i][j], E2[i][j]);
          }
          E2[rb * 4 + i][j] = En[i][j];
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
  pass1(conv_base, E2);

  for (int c = 0; c < n_chunks; c++) {
    cp_async_wait<0>();
    __syncthreads();
    convert(c + 2);
    issue(c + 3);
    if (c + 1 < n_chunks) unit(std::true_type{}, c); else unit(std::false_type{}, c);
  }
  cp_async_wait<0>();

  // ---------------- epilogue: decode, canonicalise, store ----------------
#pragma unroll
  for (int i = 0; i < 4; i++) {
    const int gm = m0 + ty * 4 + i;
    if (gm >= p.M) continue;
#pragma unroll
    for (int q = 0; q < 2; q++) {
      const int gn = n0 + q * (BN / 2) + tx * 4;
      int32_t e[4]; uint64_t c[4];
#pragma unroll
      for (int j = 0; j < 4; j++) {
        const uint32_t h = (E2[i][q * 2 + (j >> 1)] >> ((j & 1) * 16)) & 0xffffu;
        const bool fin = h >= (uint32_t)FINITE2;
        e[j] = fin ? (int32_t)h - 2 * BIAS : NEG_INF;
        uint64_t tot = (uint64_t)C[i][q * 4 + j];
        if constexpr (CM == CM_CARRY31) tot += (uint64_t)H[i][q * 4 + j] << 31;
        c[j] = fin ? tot : 0ull;
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

inline bool al16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

template <bool KM, int TB, int CM>
void launch_p16(const GemmArgs &a, int64_t batch, cudaStream_t st) {
  using G = Cfg<TB>;
  const int64_t n_cta = (int64_t)((a.N + G::BN - 1) / G::BN) * ((a.M + G::BM - 1) / G::BM) * batch * a.G;
  cudaFuncSetAttribute(gemm_pack16_kernel<KM, TB, CM>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::SMEM);
  gemm_pack16_kernel<KM, TB, CM><<<dim3((unsigned)n_cta), G::PT, G::SMEM, st>>>(a);
}

}  // namespace

// RING_U64, caller promises: finite |energy| <= 3967 (zero element exactly NEG_INF) and operand counts below
// 2^count_bits, count_bits <= 32.  32-bit accumulators when 2 * count_bits + ceil(log2 K) <= 32, else the carry form
// (count_bits <= 13) or 64-bit accumulators, both on the 64 x 64 tile.
void launch_gemm_pack16(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                        const int32_t *Ae, const uint64_t *Ac, const int32_t *Be, const uint64_t *Bc,
                        int32_t *Ce, uint64_t *Cc, int64_t sA, int64_t sB, int64_t sC, int count_bits, cudaStream_t st) {
  GemmArgs a{G, M, N, K, Ae, Ac, Be, Bc, Ce, Cc, sA, sB, sC, 0, 0, 0};
  const int ldA = a_kmajor ? M : K;
  a.vecA = (ldA % 4 == 0) && (sA % 4 == 0) && (((int64_t)M * K) % 4 == 0 || G == 1) && al16(Ae) && al16(Ac);
  a.vecB = (N % 4 == 0) && (sB % 4 == 0) && (((int64_t)K * N) % 4 == 0 || G == 1) && al16(Be) && al16(Bc);
  a.vecC = (N % 4 == 0) && (sC % 4 == 0) && (((int64_t)M * N) % 4 == 0 || G == 1) && al16(Ce) && al16(Cc);
  // the 64 x 64 tile: where a 128-row tile would be >= 75 % padding, and where 128 x 128 tiles would leave SMs idle
  // (fewer tiles than SMs: four times as many small tiles fill the machine better than the big tile's efficiency costs)
  const int64_t n_cta128 = (int64_t)((M + 127) / 128) * ((N + 127) / 128) * batch * G;
  const bool small = (M <= 64 && N <= 64) || n_cta128 < 148;
  int lgK = 0;
  while (((int64_t)1 << lgK) < K) lgK++;
  const int cm = (count_bits <= 16 && 2 * count_bits + lgK <= 32) ? CM_ACC32 : (count_bits <= 13 ? CM_CARRY31 : CM_WIDE64);
  if (cm == CM_ACC32) {
    if (a_kmajor) { if (small) launch_p16<true, 64, CM_ACC32>(a, batch, st); else launch_p16<true, 128, CM_ACC32>(a, batch, st); }
    else { if (small) launch_p16<false, 64, CM_ACC32>(a, batch, st); else launch_p16<false, 128, CM_ACC32>(a, batch, st); }
  } else if (cm == CM_CARRY31) {
    if (a_kmajor) launch_p16<true, 64, CM_CARRY31>(a, batch, st); else launch_p16<false, 64, CM_CARRY31>(a, batch, st);
  } else {
    if (a_kmajor) launch_p16<true, 64, CM_WIDE64>(a, batch, st); else launch_p16<false, 64, CM_WIDE64>(a, batch, st);
  }
}

}  // namespace bbtn
