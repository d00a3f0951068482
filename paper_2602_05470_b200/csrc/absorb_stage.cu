// absorb_stage.cu -- K3, streaming form, for a MID-SIZED gathered operand (sm_100a).
//
//   C[b][o] = (+)_k A[b][fa(o) + ka(k)] (.) B[b][fb(o) + kb(k)]      (PAPER.md:51 Eq. 2 pairwise, :57)
//
// absorb_vec.cu reads B straight from global memory: fine while B is a bond or vertex tensor (a few elements, always in
// L1), but in balanced trees B has hundreds or thousands of elements, every fold of every vector waits for 8-16
// dependent L1/L2 loads, and the write-heavy nodes that grow a tensor (2^17 (x) 2^13 -> 2^20 elements per leaf on the
// 5x5x5 cube) ran at 3.7-4.8 TB/s with the schedulers idle half the time (long-scoreboard stalls).  Here the elements
// of B that ONE TILE of 4096 x 2^NF outputs can meet -- B's bits among the tile's low output bits, the summed bit and
// the folded new legs: at most 2048 elements -- are first gathered into shared memory in a compact layout (coalesced
// when the planner has re-laid B in output order, plan.cpp), and the inner loop reads them from there.
// Same thread mapping as absorb_vec.cu's LP_FAR case: a thread owns 4 consecutive outputs (16-byte loads of A,
// 16-byte stores of C) and produces all 2^NF folded outputs that share an element of A from one read of A.
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

struct StageArgs {
  int rO, nK, tb, fbits;          // rank of the output WITHOUT its folded top bits, summed bits (0 or 1), tile bits, log2 footprint
  uint32_t addA[32], addB[32];    // per output bit (global element offsets)
  uint32_t kA;                    // offset into A of the summed bit
  uint32_t sg[12];                // compact bit c of the staged footprint -> offset into B
  uint32_t sadd[12];              // output bit q < tb -> compact offset (0 where B does not carry it)
  uint32_t sk, sfold[4];          // compact offset of the summed bit and of each combination of the folded bits
  int64_t sA, sB, sC, n_tiles;    // batch strides (elements), tiles over all batch entries
  int b_unit;                     // B's counts are all 0/1: the product of the counts is A's count
};

template <class CT> struct V4;
template <> struct V4<uint64_t> {
  uint64_t v[4];
  __device__ __forceinline__ void load(const uint64_t *p) {
    asm("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(v[0]), "=l"(v[1]), "=l"(v[2]), "=l"(v[3]) : "l"(p));
  }
  __device__ __forceinline__ void store(uint64_t *p) const {
    asm volatile("st.global.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(v[0]), "l"(v[1]), "l"(v[2]), "l"(v[3]));
  }
};
template <> struct V4<NoCount> {
  NoCount v[4];
  __device__ __forceinline__ void load(const NoCount *) {}
  __device__ __forceinline__ void store(NoCount *) const {}
};

__device__ __forceinline__ void load_e4(const int32_t *p, int32_t *d) {
  const int4 a = *reinterpret_cast<const int4 *>(p);
  d[0] = a.x; d[1] = a.y; d[2] = a.z; d[3] = a.w;
}

// BV: how the 4 outputs of a vector meet the staged B.  1: all four read the same element (B carries neither of the two
// lowest output bits); 2: four consecutive elements (it carries both: they are compact bits 0 and 1) -- one 16-byte and
// two 16-byte shared-memory reads instead of eight scalar ones; 3 / 4: two consecutive elements chosen by output bit 0 /
// bit 1 (it carries only that one); 0: anything else.
template <class CT> __device__ __forceinline__ void lds_c4(const CT *p, CT *d);
template <> __device__ __forceinline__ void lds_c4<uint64_t>(const uint64_t *p, uint64_t *d) {
  const ulonglong2 a = *reinterpret_cast<const ulonglong2 *>(p), b = *reinterpret_cast<const ulonglong2 *>(p + 2);
  d[0] = a.x; d[1] = a.y; d[2] = b.x; d[3] = b.y;
}
template <> __device__ __forceinline__ void lds_c4<NoCount>(const NoCount *, NoCount *) {}

template <class R, int NF, int BV>
__global__ void __launch_bounds__(256) absorb_stage_kernel(StageArgs p, const int32_t *__restrict__ Ae,
                                                           const typename R::T *__restrict__ Ac,
                                                           const int32_t *__restrict__ Be, const typename R::T *__restrict__ Bc,
                                                           int32_t *__restrict__ Ce, typename R::T *__restrict__ Cc) {
  using CT = typename R::T;
  constexpr int VPT = 4, NFV = 1 << NF;
  extern __shared__ __align__(16) unsigned char smem[];
  const int foot = 1 << p.fbits;
  int32_t *sBe = reinterpret_cast<int32_t *>(smem);
  CT *sBc = reinterpret_cast<CT *>(smem + ((4 * foot + 15) & ~15));      // (unused by the count-free ring)
  const int nvec = 1 << (p.tb - 2);
  uint32_t ta[VPT], ts[VPT];                               // per-thread part of the addresses: output bits 2 .. tb-1
#pragma unroll
  for (int j = 0; j < VPT; j++) {
    const uint32_t o = (uint32_t)(threadIdx.x + 256 * j) << 2;
    uint32_t a = 0, s = 0;
    for (int q = 2; q < p.tb; q++) if ((o >> q) & 1u) { a += p.addA[q]; s += p.sadd[q]; }
    ta[j] = a; ts[j] = s;
  }
  const uint32_t us1 = p.sadd[0], us2 = p.sadd[1];
  const int tiles_per_entry_lg = p.rO - p.tb;
  const int n_k = 1 << p.nK;

  for (int64_t t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
    const int64_t b = t >> tiles_per_entry_lg;
    const uint32_t hi = (uint32_t)(t - (b << tiles_per_entry_lg));
    uint32_t a_hi = 0, b_hi = 0;
    for (int q = 0; q < tiles_per_entry_lg; q++) if ((hi >> q) & 1u) { a_hi += p.addA[p.tb + q]; b_hi += p.addB[p.tb + q]; }
    const int32_t *ae = Ae + b * p.sA + a_hi; const CT *ac = Ac + b * p.sA + a_hi;
    const int32_t *be = Be + b * p.sB + b_hi; const CT *bc = Bc + b * p.sB + b_hi;
    int32_t *ce = Ce + b * p.sC + ((int64_t)hi << p.tb); CT *cc = Cc + b * p.sC + ((int64_t)hi << p.tb);
    // ---- the tile's footprint in B -> shared memory, compact
    __syncthreads();                                       // the previous tile's readers are done
    for (int i = threadIdx.x; i < foot; i += 256) {
      uint32_t off = 0;
      for (int q = 0; q < p.fbits; q++) if ((i >> q) & 1) off += p.sg[q];
      sBe[i] = be[off];
      stc<R>(sBc, i, ldc<R>(bc, off));
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < VPT; j++) {
      const int v = threadIdx.x + 256 * j;
      if (v >= nvec) break;
      int32_t e4[2][4]; V4<CT> c4[2];
      load_e4(ae + ta[j], e4[0]); c4[0].load(ac + ta[j]);
      if (p.nK == 1) { load_e4(ae + ta[j] + p.kA, e4[1]); c4[1].load(ac + ta[j] + p.kA); }
#pragma unroll
      for (int f = 0; f < NFV; f++) {
        int32_t acc_e[4]; CT acc_c[4];
        const uint32_t sf = ts[j] + p.sfold[f];
#pragma unroll
        for (int k = 0; k < 2; k++) {
          if (k < n_k) {
            const uint32_t sk = sf + (k ? p.sk : 0u);
            int32_t eb[4]; CT cb[4];
            if (BV == 1) {
              eb[0] = eb[1] = eb[2] = eb[3] = sBe[sk];
              if (!p.b_unit) cb[0] = cb[1] = cb[2] = cb[3] = ldc<R>(sBc, sk);
            } else if (BV == 2) {
              load_e4(sBe + sk, eb);
              if (!p.b_unit) lds_c4<CT>(sBc + sk, cb);
            } else if (BV == 3 || BV == 4) {               // two consecutive elements, selected by output bit 0 (3) or bit 1 (4)
              const int2 e2 = *reinterpret_cast<const int2 *>(sBe + sk);
              CT c2[2];
              if (!p.b_unit) { c2[0] = ldc<R>(sBc, sk); c2[1] = ldc<R>(sBc, sk + 1); }
#pragma unroll
              for (int u = 0; u < 4; u++) {
                const int sel = BV == 3 ? (u & 1) : (u >> 1);
                eb[u] = sel ? e2.y : e2.x;
                if (!p.b_unit) cb[u] = c2[sel];
              }
            } else {
#pragma unroll
              for (int u = 0; u < 4; u++) {
                const uint32_t is = sk + ((u & 1) ? us1 : 0u) + ((u & 2) ? us2 : 0u);
                eb[u] = sBe[is];
                if (!p.b_unit) cb[u] = ldc<R>(sBc, is);
              }
            }
            // the first term is taken as it is (a sum below -2^29 is canonicalised to the zero element at the end, exactly as
            // (+) with the zero element would have left it), the second one is (+)-merged
#pragma unroll
            for (int u = 0; u < 4; u++) {
              const int32_t e = e4[k][u] + eb[u];
              const CT c = p.b_unit ? c4[k].v[u] : R::mul(c4[k].v[u], cb[u]);
              if (k == 0) { acc_e[u] = e; acc_c[u] = c; } else oplus<R>(acc_e[u], acc_c[u], e, c);
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
    }
  }
}

inline bool al16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }
inline bool al32(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 31) == 0; }

}  // namespace

// Returns false when the step does not fit this form (the caller then tries absorb_vec.cu, then the scalar kernel).
bool launch_absorb_stage(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                         int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs) {
  if (xs || s.n_slice || s.xA || s.xB) return false;                   // dense operands only
  if (s.rB < 7 || s.rO < 14 || s.nK > 1 || s.rA < 3) return false;     // a mid-sized B under a large output
  if (!(s.addA[0] == 1u && s.addA[1] == 2u)) return false;             // the 4 outputs of a vector are 4 consecutive elements of A
  if (s.nK == 1 && s.kA[0] < 4u) return false;
  if (!al16(Ae) || !al16(Ce) || (ring != RING_NONE && (!al32(Ac) || !al32(Cc)))) return false;
  int nF = 0;                                                          // fold the top output bits that only B carries
  while (nF < 2 && s.rO - nF > 4 && s.addA[s.rO - 1 - nF] == 0u) nF++;
  const int rOe = s.rO - nF;
  for (int q = 2; q < s.rO; q++) if (s.addA[q] & 3u) return false;     // the 16-byte reads of A stay aligned
  StageArgs p;
  p.rO = rOe; p.nK = s.nK; p.tb = rOe < 12 ? rOe : 12;
  for (int i = 0; i < 32; i++) { p.addA[i] = s.addA[i]; p.addB[i] = s.addB[i]; }
  p.kA = s.nK ? s.kA[0] : 0u;
  // compact layout of the footprint: B's bits among the tile's output bits (in output order), the summed bit, the folded bits
  int c = 0;
  for (int q = 0; q < 12; q++) { p.sg[q] = 0; p.sadd[q] = 0; }
  for (int q = 0; q < p.tb; q++) if (s.addB[q]) { if (c >= 11) return false; p.sadd[q] = 1u << c; p.sg[c] = s.addB[q]; c++; }
  p.sk = 0;
  if (s.nK) { if (c >= 11) return false; p.sk = 1u << c; p.sg[c] = s.kB[0]; c++; }
  int fold_bit[2] = {0, 0};
  for (int i = 0; i < nF; i++) { if (c >= 11) return false; fold_bit[i] = c; p.sg[c] = s.addB[rOe + i]; c++; }
  for (int f = 0; f < 4; f++) { p.sfold[f] = 0; for (int i = 0; i < nF; i++) if ((f >> i) & 1) p.sfold[f] += 1u << fold_bit[i]; }
  p.fbits = c;
  if (c > 11 || ((int64_t)1 << (p.tb + nF)) < ((int64_t)8 << c)) return false;     // each staged element must serve >= 8 outputs
  p.sA = s.vA ? ((int64_t)1 << s.rA) : 0;
  p.sB = s.vB ? ((int64_t)1 << s.rB) : 0;
  p.sC = (int64_t)1 << s.rO;
  p.b_unit = s.b_unit;
  p.n_tiles = nb << (rOe - p.tb);
  const int64_t cap = 148 * 8;
  const int grid = (int)(p.n_tiles < cap ? p.n_tiles : cap);
  const size_t smem = ((((size_t)4 << c) + 15) & ~(size_t)15) + (ring_count_bytes(ring) << c);
  const int bv = (p.sadd[0] == 0u && p.sadd[1] == 0u) ? 1 : (p.sadd[0] == 1u && p.sadd[1] == 2u) ? 2
                 : (p.sadd[0] == 1u && p.sadd[1] == 0u) ? 3 : (p.sadd[0] == 0u && p.sadd[1] == 1u) ? 4 : 0;
#define BBTN_STAGE_LAUNCH(NFV_, BV_)                                                                                \
  absorb_stage_kernel<R, NFV_, BV_><<<grid, 256, smem, st>>>(p, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc)
#define BBTN_STAGE_NF(BV_)                                                                                          \
  do { if (nF == 0) BBTN_STAGE_LAUNCH(0, BV_); else if (nF == 1) BBTN_STAGE_LAUNCH(1, BV_); else BBTN_STAGE_LAUNCH(2, BV_); } while (0)
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    if (bv == 1) BBTN_STAGE_NF(1); else if (bv == 2) BBTN_STAGE_NF(2); else if (bv == 3) BBTN_STAGE_NF(3);
    else if (bv == 4) BBTN_STAGE_NF(4); else BBTN_STAGE_NF(0);
  });
#undef BBTN_STAGE_NF
#undef BBTN_STAGE_LAUNCH
  return true;
}

}  // namespace bbtn
