// absorb_vec.cu -- K3, streaming form, vectorised (sm_100a).
//
//   C[b][o] = (+)_k A[b][fa(o) + ka(k)] (.) B[b][fb(o) + kb(k)]      (PAPER.md:51 Eq. 2 pairwise, :57)
//
// This is the HBM-bound shape of the pairwise contraction: a large tensor A absorbs a small one (a bond
// or vertex tensor, or a narrow intermediate) and at most a few indices are summed, so there is ~1/12
// tropical FMA per byte and the kernel has to move 12 B per element at memory speed.  The planner lays
// the output out as "A's surviving bits in A's order, then B's new bits", so runs of consecutive outputs
// are runs of consecutive (or regularly interleaved) elements of A:
//   * a thread owns 4 consecutive outputs: 16-byte loads of A, 16-byte stores of C;
//   * fa/fb are sums of per-bit offsets (all dims are 2), split into a per-thread part (bits 2..11,
//     computed once), and a per-tile part (bits >= 12, a short loop per 4096 outputs);
//   * the three ways the lowest two output bits can sit in A are compile-time cases (LP): both are A's
//     bits 0,1 (FAR: the summed index lies higher), or the summed index is A's bit 0 (K0) or bit 1 (K1),
//     in which case one 8-element read holds both k for all 4 outputs.
// Anything else (rank < 4, several summed low bits, unaligned arena offsets) takes the scalar kernel.
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

enum LowPattern : int { LP_FAR = 0, LP_K0 = 1, LP_K1 = 2 };

struct AbsorbVecArgs {
  int rO, nK, tb;                 // rank of the output WITHOUT its folded top bits, summed bits, tile bits (<= 12)
  uint32_t foldB[4];              // offset into B of each combination of the folded (new, B-only) top output bits
  uint32_t addA[32], addB[32];    // per output bit
  uint32_t kA[8], kB[8];          // per summed bit
  int64_t sA, sB, sC, n_tiles;    // batch strides (elements), tiles over all batch entries
  int b_unit;                     // B's counts are all 0/1: the product of the counts is A's count (Step::b_unit)
  const uint8_t *xs; int nF;      // local slicing: rows [nb][nF] of 0/1 and the strides of the fixed indices
  uint32_t sliceA[24], sliceB[24];
};

template <class CT> struct V4;
template <> struct V4<uint64_t> {
  uint64_t v[4];
  // 32-byte global accesses (LDG.E.256 / STG.E.256, new on sm_100): one full 32-byte sector per thread instead
  // of two half-filled ones per instruction
  __device__ __forceinline__ void load(const uint64_t *p) {
    asm("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(v[0]), "=l"(v[1]), "=l"(v[2]), "=l"(v[3]) : "l"(p));
  }
  __device__ __forceinline__ void store(uint64_t *p) const {
    asm volatile("st.global.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(v[0]), "l"(v[1]), "l"(v[2]), "l"(v[3]));
  }
};
template <> struct V4<uint32_t> {
  uint32_t v[4];
  __device__ __forceinline__ void load(const uint32_t *p) {
    const uint4 a = *reinterpret_cast<const uint4 *>(p);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
  }
  __device__ __forceinline__ void store(uint32_t *p) const { *reinterpret_cast<uint4 *>(p) = make_uint4(v[0], v[1], v[2], v[3]); }
};

template <> struct V4<NoCount> {                 // search mode: no count plane
  NoCount v[4];
  __device__ __forceinline__ void load(const NoCount *) {}
  __device__ __forceinline__ void store(NoCount *) const {}
};

__device__ __forceinline__ void load_e4(const int32_t *p, int32_t *d) {
  const int4 a = *reinterpret_cast<const int4 *>(p);
  d[0] = a.x; d[1] = a.y; d[2] = a.z; d[3] = a.w;
}

// NF = number of FOLDED output bits: the planner puts the indices that only B carries (the new legs) at the
// top of the output, where A's address does not depend on them.  One thread produces all 2^NF outputs that
// share an element of A from a single read of A -- otherwise a node that grows the tensor reads A 2^NF times
// from DRAM (the re-reads lie 2^(rO-NF) elements apart, far beyond any cache).
template <class R, int LP, int NF>
__global__ void __launch_bounds__(256) absorb_vec_kernel(AbsorbVecArgs p, const int32_t *__restrict__ Ae,
                                                         const typename R::T *__restrict__ Ac,
                                                         const int32_t *__restrict__ Be, const typename R::T *__restrict__ Bc,
                                                         int32_t *__restrict__ Ce, typename R::T *__restrict__ Cc) {
  using CT = typename R::T;
  constexpr int VPT = 4;                                    // vectors per thread in a full 4096-output tile
  constexpr int NFV = 1 << NF;
  const int nvec = 1 << (p.tb - 2);
  // per-thread part of the addresses: output bits 2 .. tb-1
  uint32_t ta[VPT], tbo[VPT];
#pragma unroll
  for (int j = 0; j < VPT; j++) {
    const uint32_t o = (uint32_t)(threadIdx.x + 256 * j) << 2;
    uint32_t a = 0, b = 0;
    for (int q = 2; q < p.tb; q++) if ((o >> q) & 1u) { a += p.addA[q]; b += p.addB[q]; }
    ta[j] = a; tbo[j] = b;
  }
  const uint32_t ub1 = p.addB[0], ub2 = p.addB[1];
  const int tiles_per_entry_lg = p.rO - p.tb;
  const int n_k = 1 << p.nK;
  uint32_t fb[NFV];
#pragma unroll
  for (int f = 0; f < NFV; f++) fb[f] = p.foldB[f];

  for (int64_t t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
    const int64_t b = t >> tiles_per_entry_lg;
    const uint32_t hi = (uint32_t)(t - (b << tiles_per_entry_lg));
    uint32_t a_hi = 0, b_hi = 0;
    for (int q = 0; q < tiles_per_entry_lg; q++) if ((hi >> q) & 1u) { a_hi += p.addA[p.tb + q]; b_hi += p.addB[p.tb + q]; }
    int64_t oA = b * p.sA + a_hi, oB = b * p.sB + b_hi;
    if (p.nF) {
      const uint8_t *x = p.xs + b * p.nF;
      for (int j = 0; j < p.nF; j++) if (x[j]) { oA += p.sliceA[j]; oB += p.sliceB[j]; }
    }
    const int32_t *ae = Ae + oA; const CT *ac = Ac + oA;
    const int32_t *be = Be + oB; const CT *bc = Bc + oB;
    int32_t *ce = Ce + b * p.sC + ((int64_t)hi << p.tb); CT *cc = Cc + b * p.sC + ((int64_t)hi << p.tb);
#pragma unroll
    for (int j = 0; j < VPT; j++) {
      const int v = threadIdx.x + 256 * j;
      if (v >= nvec) break;
      if (LP == LP_FAR) {
        // A's vector(s) stay in registers for nK <= 1 (the common case); the folded combinations run one at a time.
        // With more summed bits and folded bits (rare) A is simply re-read per combination (L1/L2 hits, no DRAM traffic).
        const bool in_regs = NF > 0 && p.nK <= 1;      // nothing folded: stream A per k, fewest registers
        int32_t e4[2][4]; V4<CT> c4[2];
        if (in_regs) {
          load_e4(ae + ta[j], e4[0]); c4[0].load(ac + ta[j]);
          if (p.nK == 1) { load_e4(ae + ta[j] + p.kA[0], e4[1]); c4[1].load(ac + ta[j] + p.kA[0]); }
        }
#pragma unroll 1
        for (int f = 0; f < NFV; f++) {
          int32_t acc_e[4]; CT acc_c[4];
          const uint32_t fbf = p.foldB[f];
#pragma unroll
          for (int u = 0; u < 4; u++) { acc_e[u] = NEG_INF; acc_c[u] = czero<R>(); }
          if (in_regs) {
#pragma unroll
            for (int k = 0; k < 2; k++) {
              if (k < n_k) {
                const uint32_t kb = k ? p.kB[0] : 0u;
#pragma unroll
                for (int u = 0; u < 4; u++) {
                  const uint32_t ib = tbo[j] + kb + fbf + ((u & 1) ? ub1 : 0u) + ((u & 2) ? ub2 : 0u);
                  const int32_t e = e4[k][u] + be[ib];
                  const CT c = p.b_unit ? c4[k].v[u] : R::mul(c4[k].v[u], ldc<R>(bc, ib));
                  // the first term is taken as it is (a sum below -2^29 is canonicalised to the zero element below, exactly
                  // as (+) with the zero element would have left it), the second one is (+)-merged
                  if (k == 0) { acc_e[u] = e; acc_c[u] = c; } else oplus<R>(acc_e[u], acc_c[u], e, c);
                }
              }
            }
          } else {
            for (int k = 0; k < n_k; k++) {
              uint32_t ka = 0, kb = 0;
              for (int q = 0; q < p.nK; q++) if ((k >> q) & 1) { ka += p.kA[q]; kb += p.kB[q]; }
              int32_t ex[4]; V4<CT> cx;
              load_e4(ae + ta[j] + ka, ex); cx.load(ac + ta[j] + ka);
#pragma unroll
              for (int u = 0; u < 4; u++) {
                const uint32_t ib = tbo[j] + kb + fbf + ((u & 1) ? ub1 : 0u) + ((u & 2) ? ub2 : 0u);
                oplus<R>(acc_e[u], acc_c[u], ex[u] + be[ib], p.b_unit ? cx.v[u] : R::mul(cx.v[u], ldc<R>(bc, ib)));
              }
            }
          }
          V4<CT> oc;
#pragma unroll
          for (int u = 0; u < 4; u++) { canonicalise<R>(acc_e[u], acc_c[u]); oc.v[u] = acc_c[u]; }
          const int64_t fo = ((int64_t)f << p.rO) + 4 * v;
          *reinterpret_cast<int4 *>(ce + fo) = make_int4(acc_e[0], acc_e[1], acc_e[2], acc_e[3]);
          oc.store(cc + fo);
        }
      } else {
        // nK == 1 and the summed index is A's bit 0 (K0) or bit 1 (K1): 8 consecutive elements of A hold both k of
        // all 4 outputs.  One folded combination at a time (not unrolled: unrolling hoists the 16 B-operand loads
        // of every combination and costs 178 registers, one CTA per SM)
        int32_t e8[8]; V4<CT> c8[2];
        load_e4(ae + ta[j], e8); load_e4(ae + ta[j] + 4, e8 + 4);
        c8[0].load(ac + ta[j]); c8[1].load(ac + ta[j] + 4);
#pragma unroll 1
        for (int f = 0; f < NFV; f++) {
          int32_t acc_e[4]; CT acc_c[4];
          const uint32_t fbf = p.foldB[f];
#pragma unroll
          for (int u = 0; u < 4; u++) {
#pragma unroll
            for (int k = 0; k < 2; k++) {
              // element index inside the 8: K0: 2u + k;  K1: (u & 1) + 2k + 4(u >> 1)
              const int idx = LP == LP_K0 ? 2 * u + k : (u & 1) + 2 * k + 4 * (u >> 1);
              const uint32_t ib = tbo[j] + fbf + (k ? p.kB[0] : 0u) + ((u & 1) ? ub1 : 0u) + ((u & 2) ? ub2 : 0u);
              const int32_t e = e8[idx] + be[ib];
              const CT c = p.b_unit ? c8[idx >> 2].v[idx & 3] : R::mul(c8[idx >> 2].v[idx & 3], ldc<R>(bc, ib));
              if (k == 0) { acc_e[u] = e; acc_c[u] = c; } else oplus<R>(acc_e[u], acc_c[u], e, c);      // (first term assigned, as above)
            }
          }
          V4<CT> oc;
#pragma unroll
          for (int u = 0; u < 4; u++) { canonicalise<R>(acc_e[u], acc_c[u]); oc.v[u] = acc_c[u]; }
          const int64_t fo = ((int64_t)f << p.rO) + 4 * v;
          *reinterpret_cast<int4 *>(ce + fo) = make_int4(acc_e[0], acc_e[1], acc_e[2], acc_e[3]);
          oc.store(cc + fo);
        }
      }
    }
  }
}

inline bool al16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }
inline bool al32(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 31) == 0; }

}  // namespace

// Returns false when the step does not fit the vectorised form (the caller then runs the scalar kernel).
bool launch_absorb_vec(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                       int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs) {
  if (s.rO < 4 || s.nK > 3 || s.rA < 3) return false;
  if (xs) for (int j = 0; j < s.n_slice; j++) if (s.sliceA[j] & 3u) return false;   // a slice would break the 16-byte reads of A
  if (!al16(Ae) || !al16(Ce) || (ring != RING_NONE && (!al16(Ac) || !al16(Cc)))) return false;
  if (ring_count_bytes(ring) == 8 && (!al32(Ac) || !al32(Cc))) return false;       // 32-byte count vectors
  int lp;
  if (s.addA[0] == 1u && s.addA[1] == 2u) {
    lp = LP_FAR;
    for (int q = 0; q < s.nK; q++) if (s.kA[q] < 4u) return false;
  } else if (s.nK == 1 && s.kA[0] == 1u && s.addA[0] == 2u && s.addA[1] == 4u) lp = LP_K0;
  else if (s.nK == 1 && s.kA[0] == 2u && s.addA[0] == 1u && s.addA[1] == 4u) lp = LP_K1;
  else return false;
  // fold the top output bits that only B carries (see the kernel comment); keep >= 4 unfolded bits
  int nF = 0;
  while (nF < 2 && s.rO - nF > 4 && s.addA[s.rO - 1 - nF] == 0u) nF++;
  const int rOe = s.rO - nF;
  AbsorbVecArgs p;
  p.rO = rOe; p.nK = s.nK; p.tb = rOe < 12 ? rOe : 12;
  for (int i = 0; i < 32; i++) { p.addA[i] = s.addA[i]; p.addB[i] = s.addB[i]; }
  for (int i = 0; i < 8; i++) { p.kA[i] = s.kA[i]; p.kB[i] = s.kB[i]; }
  for (int f = 0; f < 4; f++) {
    p.foldB[f] = 0;
    for (int i = 0; i < nF; i++) if ((f >> i) & 1) p.foldB[f] += s.addB[rOe + i];
  }
  // the 16-byte reads of A must stay 4-element aligned: every offset that can be added is a multiple of 4
  for (int q = 2; q < s.rO; q++) if (p.addA[q] & 3u) return false;
  p.sA = (s.vA && !s.xA) ? ((int64_t)1 << s.rA) : 0;
  p.sB = (s.vB && !s.xB) ? ((int64_t)1 << s.rB) : 0;
  p.sC = (int64_t)1 << s.rO;
  p.b_unit = s.b_unit;
  p.xs = xs; p.nF = xs ? s.n_slice : 0;
  for (int j = 0; j < 24; j++) { p.sliceA[j] = s.sliceA[j]; p.sliceB[j] = s.sliceB[j]; }
  p.n_tiles = nb << (rOe - p.tb);
  const int64_t cap = 148 * 8;
  const int grid = (int)(p.n_tiles < cap ? p.n_tiles : cap);
#define BBTN_ABSORB_LAUNCH(LPV, NFV_)                                                                               \
  absorb_vec_kernel<R, LPV, NFV_><<<grid, 256, 0, st>>>(p, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc)
#define BBTN_ABSORB_NF(LPV)                                                                                         \
  do { if (nF == 0) BBTN_ABSORB_LAUNCH(LPV, 0); else if (nF == 1) BBTN_ABSORB_LAUNCH(LPV, 1); else BBTN_ABSORB_LAUNCH(LPV, 2); } while (0)
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    if (lp == LP_FAR) BBTN_ABSORB_NF(LP_FAR);
    else if (lp == LP_K0) BBTN_ABSORB_NF(LP_K0);
    else BBTN_ABSORB_NF(LP_K1);
  });
#undef BBTN_ABSORB_NF
#undef BBTN_ABSORB_LAUNCH
  return true;
}

}  // namespace bbtn
