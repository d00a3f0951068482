// kernels.cu -- K1 construct, K3 streaming/long-reduction forms, K4 finalize (sm_100a).
#include "kernels.h"
#include "ring.cuh"
#include "construct.cuh"
#include <type_traits>

namespace bbtn {
namespace {

template <class R>
__global__ void construct_tensors_kernel(int kind, const InputRec *__restrict__ inputs, const int32_t *__restrict__ list,
                                         int n_list, const uint8_t *__restrict__ assign, int n_fixed, int64_t B,
                                         int32_t *__restrict__ out_e, typename R::T *__restrict__ out_c) {
  const int64_t total = B * n_list;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t b = t / n_list;
    const InputRec r = inputs[list[t - b * n_list]];
    const int fu_val = r.fu >= 0 ? assign[b * n_fixed + r.fu] : 0;
    const int fv_val = r.fv >= 0 ? assign[b * n_fixed + r.fv] : 0;
    const int n_el = 1 << r.rank;
    const int64_t base = r.offset * B + b * n_el;
    for (int x = 0; x < n_el; x++) {
      int xu = r.bu >= 0 ? (x >> r.bu) & 1 : 0;
      int xv = r.bv >= 0 ? (x >> r.bv) & 1 : 0;
      int32_t e; typename R::T c;
      input_element<R>(kind, r, fu_val, fv_val, xu, xv, e, c);
      out_e[base + x] = e;
      stc<R>(out_c, base + x, c);
    }
  }
}

// offset[b] = (.) over every rank-0 input of leaf b (fully fixed bonds, fixed vertices, isolated vertices)
template <class R>
__global__ void construct_offset_kernel(int kind, const InputRec *__restrict__ inputs, const int32_t *__restrict__ list,
                                        int n_list, const uint8_t *__restrict__ assign, int n_fixed, int64_t B,
                                        int32_t *__restrict__ off_e, typename R::T *__restrict__ off_c) {
  for (int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; b < B; b += (int64_t)gridDim.x * blockDim.x) {
    int32_t acc_e = 0; typename R::T acc_c = R::from_small(1);
    for (int i = 0; i < n_list; i++) {
      const InputRec r = inputs[list[i]];
      const int fu_val = r.fu >= 0 ? assign[b * n_fixed + r.fu] : 0;
      const int fv_val = r.fv >= 0 ? assign[b * n_fixed + r.fv] : 0;
      int32_t e; typename R::T c;
      input_element<R>(kind, r, fu_val, fv_val, 0, 0, e, c);
      acc_e += e; acc_c = R::mul(acc_c, c);
      canonicalise<R>(acc_e, acc_c);
    }
    off_e[b] = acc_e; stc<R>(off_c, b, acc_c);
  }
}

// ---------------------------------------------------------------------------------------------
// K3, streaming form: one thread per output element, the bit permutation of both operands is folded
// into the address computation (no separate K2 pass):  C[o] = (+)_k A[fa(o)+ka(k)] (.) B[fb(o)+kb(k)].
// ---------------------------------------------------------------------------------------------
struct AbsorbArgs {
  int rO, nK;
  uint32_t addA[32], addB[32], kA[32], kB[32];
  int64_t sA, sB, sC, total;
  const uint8_t *xs; int nF;               // local slicing: rows [nb][nF] of 0/1 and the strides of the fixed indices
  uint32_t sliceA[24], sliceB[24];
};

// element offset of batch entry b's operands: b * stride, plus the strides of the locally fixed indices that are set
template <class ARGS>
__device__ __forceinline__ void batch_offsets(const ARGS &p, int64_t b, int64_t &oA, int64_t &oB) {
  oA = b * p.sA; oB = b * p.sB;
  if (p.nF) {
    const uint8_t *x = p.xs + b * p.nF;
    for (int j = 0; j < p.nF; j++) if (x[j]) { oA += p.sliceA[j]; oB += p.sliceB[j]; }
  }
}

template <class R>
__global__ void absorb_kernel(AbsorbArgs p, const int32_t *__restrict__ Ae, const typename R::T *__restrict__ Ac,
                              const int32_t *__restrict__ Be, const typename R::T *__restrict__ Bc,
                              int32_t *__restrict__ Ce, typename R::T *__restrict__ Cc) {
  const int64_t omask = ((int64_t)1 << p.rO) - 1;      // rO may be 32
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < p.total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t b = t >> p.rO;
    const uint32_t o = (uint32_t)(t & omask);
    uint32_t a0 = 0, b0 = 0;
    for (int q = 0; q < p.rO; q++) if ((o >> q) & 1u) { a0 += p.addA[q]; b0 += p.addB[q]; }
    int64_t oA, oB;
    batch_offsets(p, b, oA, oB);
    const int32_t *ae = Ae + oA; const typename R::T *ac = Ac + oA;
    const int32_t *be = Be + oB; const typename R::T *bc = Bc + oB;
    int32_t acc_e = NEG_INF; typename R::T acc_c = czero<R>();
    for (uint64_t k = 0; k < (1ull << p.nK); k++) {        // nK may be 32
      uint32_t ia = a0, ib = b0;
      for (int j = 0; j < p.nK; j++) if ((k >> j) & 1ull) { ia += p.kA[j]; ib += p.kB[j]; }
      const int32_t e = ae[ia] + be[ib];
      const typename R::T c = R::mul(ldc<R>(ac, ia), ldc<R>(bc, ib));
      oplus<R>(acc_e, acc_c, e, c);
    }
    canonicalise<R>(acc_e, acc_c);
    Ce[b * p.sC + o] = acc_e;
    stc<R>(Cc, b * p.sC + o, acc_c);
  }
}

// long-reduction form: one CTA per output element, block-wide (+) over k (tree roots, traces)
struct ReduceArgs {
  int rO, nK;
  uint32_t addA[32], addB[32], kA[32], kB[32];
  int64_t sA, sB, sC;
  const uint8_t *xs; int nF;
  uint32_t sliceA[24], sliceB[24];
};

template <class R>
__global__ void reduce_kernel(ReduceArgs p, const int32_t *__restrict__ Ae, const typename R::T *__restrict__ Ac,
                              const int32_t *__restrict__ Be, const typename R::T *__restrict__ Bc,
                              int32_t *__restrict__ Ce, typename R::T *__restrict__ Cc) {
  __shared__ int32_t sh_e[32];
  __shared__ typename std::conditional<R::kCounts, typename R::T, char>::type sh_c[32];
  const int64_t t = blockIdx.x;
  const int64_t b = t >> p.rO;
  const uint32_t o = (uint32_t)t & ((1u << p.rO) - 1u);
  uint32_t a0 = 0, b0 = 0;
  for (int q = 0; q < p.rO; q++) if ((o >> q) & 1u) { a0 += p.addA[q]; b0 += p.addB[q]; }
  int64_t oA, oB;
  batch_offsets(p, b, oA, oB);
  const int32_t *ae = Ae + oA; const typename R::T *ac = Ac + oA;
  const int32_t *be = Be + oB; const typename R::T *bc = Bc + oB;
  int32_t acc_e = NEG_INF; typename R::T acc_c = czero<R>();
  for (uint64_t k = threadIdx.x; k < (1ull << p.nK); k += blockDim.x) {      // nK may be 32
    uint32_t ia = a0, ib = b0;
    for (int j = 0; j < p.nK; j++) if ((k >> j) & 1ull) { ia += p.kA[j]; ib += p.kB[j]; }
    oplus<R>(acc_e, acc_c, ae[ia] + be[ib], R::mul(ldc<R>(ac, ia), ldc<R>(bc, ib)));
  }
  // warp (+), then across warps
  for (int d = 16; d > 0; d >>= 1) {
    int32_t oe = __shfl_xor_sync(0xffffffffu, acc_e, d);
    typename R::T oc = shfl_xor_c<R>(acc_c, d);
    oplus<R>(acc_e, acc_c, oe, oc);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { sh_e[warp] = acc_e; if constexpr (R::kCounts) sh_c[warp] = acc_c; }
  __syncthreads();
  if (warp == 0) {
    const int nw = blockDim.x >> 5;
    acc_e = lane < nw ? sh_e[lane] : NEG_INF;
    if constexpr (R::kCounts) acc_c = lane < nw ? sh_c[lane] : 0;
    for (int d = 16; d > 0; d >>= 1) {
      int32_t oe = __shfl_xor_sync(0xffffffffu, acc_e, d);
      typename R::T oc = shfl_xor_c<R>(acc_c, d);
      oplus<R>(acc_e, acc_c, oe, oc);
    }
    if (lane == 0) {
      canonicalise<R>(acc_e, acc_c);
      Ce[b * p.sC + o] = acc_e;
      stc<R>(Cc, b * p.sC + o, acc_c);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// K4: result[b] = offset[b] (.) root[b], canonical, in reported units (Ising: min H = -max-plus).
// ---------------------------------------------------------------------------------------------
template <class R>
__global__ void finalize_kernel(int kind, int64_t B, const int32_t *__restrict__ root_e,
                                const typename R::T *__restrict__ root_c, int64_t root_stride,
                                const int32_t *__restrict__ off_e, const typename R::T *__restrict__ off_c,
                                int32_t *__restrict__ energy, uint64_t *__restrict__ count,
                                uint32_t *__restrict__ count_mod, int ring) {
  for (int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; b < B; b += (int64_t)gridDim.x * blockDim.x) {
    int32_t e = off_e[b]; typename R::T c = ldc<R>(off_c, b);
    if (root_e) { e += root_e[b * root_stride]; c = R::mul(c, ldc<R>(root_c, b * root_stride)); }
    canonicalise<R>(e, c);
    const bool zero = e == NEG_INF;
    if constexpr (!R::kCounts) {                       // search mode: the energy alone; the count output reads 0
      energy[b] = zero ? NEG_INF : (kind == 0 ? -e : e);
      if (count) count[b] = 0;
    } else if (ring == 0) {
      energy[b] = zero ? NEG_INF : (kind == 0 ? -e : e);
      count[b] = (uint64_t)c;
    } else if (count_mod) {                            // RING_P12: the residue mod P1 in the low word, mod P2 in the high word
      count_mod[2 * b] = (uint32_t)c; count_mod[2 * b + 1] = (uint32_t)((uint64_t)c >> 32);
    }
  }
}

// acc (+)= (+)_b offset[b] (.) slice[b]   (local slicing: the (+) over the slices of a segment)
template <class R>
__global__ void accumulate_kernel(int64_t n, int64_t nb, const int32_t *__restrict__ slice_e, const typename R::T *__restrict__ slice_c,
                                  const int32_t *__restrict__ off_e, const typename R::T *__restrict__ off_c,
                                  int32_t *__restrict__ acc_e, typename R::T *__restrict__ acc_c, int first) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    int32_t e = NEG_INF; typename R::T c = czero<R>();
    if (slice_e) {
      if (!first) { e = acc_e[i]; c = ldc<R>(acc_c, i); }
      for (int64_t b = 0; b < nb; b++) {
        int32_t se = slice_e[b * n + i] + off_e[b]; typename R::T sc = R::mul(ldc<R>(slice_c, b * n + i), ldc<R>(off_c, b));
        canonicalise<R>(se, sc);
        oplus<R>(e, c, se, sc);
      }
      canonicalise<R>(e, c);
    }
    acc_e[i] = e; stc<R>(acc_c, i, c);
  }
}

inline int grid_for(int64_t total, int block) {
  int64_t g = (total + block - 1) / block;
  const int64_t cap = 148 * 16;          // grid-stride beyond 16 CTAs per SM
  return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

}  // namespace

void launch_construct(int kind, const InputRec *d_inputs, const int32_t *d_list_var, int n_var,
                      const int32_t *d_list_inv, int n_inv, const int32_t *d_list_scalar, int n_scalar,
                      const uint8_t *d_assign, int n_fixed, int64_t B,
                      int32_t *var_e, void *var_c, int32_t *inv_e, void *inv_c,
                      int32_t *off_e, void *off_c, int ring, cudaStream_t st) {
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    if (n_var > 0)
      construct_tensors_kernel<R><<<grid_for(B * n_var, 256), 256, 0, st>>>(kind, d_inputs, d_list_var, n_var, d_assign,
                                                                            n_fixed, B, var_e, (CT *)var_c);
    if (n_inv > 0)
      construct_tensors_kernel<R><<<grid_for(n_inv, 256), 256, 0, st>>>(kind, d_inputs, d_list_inv, n_inv, d_assign,
                                                                        n_fixed, 1, inv_e, (CT *)inv_c);
    construct_offset_kernel<R><<<grid_for(B, 128), 128, 0, st>>>(kind, d_inputs, d_list_scalar, n_scalar, d_assign,
                                                                 n_fixed, B, off_e, (CT *)off_c);
  });
}

void launch_absorb(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                   int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs) {
  if (launch_absorb_stage(s, nb, Ae, Ac, Be, Bc, Ce, Cc, ring, st, xs)) return; // mid-sized B staged in shared memory (absorb_stage.cu)
  if (launch_absorb_vec(s, nb, Ae, Ac, Be, Bc, Ce, Cc, ring, st, xs)) return;   // 16-byte form (absorb_vec.cu)
  AbsorbArgs p;
  p.rO = s.rO; p.nK = s.nK;
  for (int i = 0; i < 32; i++) { p.addA[i] = s.addA[i]; p.addB[i] = s.addB[i]; p.kA[i] = s.kA[i]; p.kB[i] = s.kB[i]; }
  p.sA = (s.vA && !s.xA) ? ((int64_t)1 << s.rA) : 0;
  p.sB = (s.vB && !s.xB) ? ((int64_t)1 << s.rB) : 0;
  p.xs = xs; p.nF = xs ? s.n_slice : 0;
  for (int j = 0; j < 24; j++) { p.sliceA[j] = s.sliceA[j]; p.sliceB[j] = s.sliceB[j]; }
  p.sC = (int64_t)1 << s.rO;
  p.total = nb << s.rO;
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    absorb_kernel<R><<<grid_for(p.total, 256), 256, 0, st>>>(p, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc);
  });
}

void launch_reduce(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                   int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs) {
  ReduceArgs p;
  p.rO = s.rO; p.nK = s.nK;
  for (int i = 0; i < 32; i++) { p.addA[i] = s.addA[i]; p.addB[i] = s.addB[i]; p.kA[i] = s.kA[i]; p.kB[i] = s.kB[i]; }
  p.sA = (s.vA && !s.xA) ? ((int64_t)1 << s.rA) : 0;
  p.sB = (s.vB && !s.xB) ? ((int64_t)1 << s.rB) : 0;
  p.xs = xs; p.nF = xs ? s.n_slice : 0;
  for (int j = 0; j < 24; j++) { p.sliceA[j] = s.sliceA[j]; p.sliceB[j] = s.sliceB[j]; }
  p.sC = (int64_t)1 << s.rO;
  const int64_t total = nb << s.rO;
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    reduce_kernel<R><<<(unsigned)total, 256, 0, st>>>(p, Ae, (const CT *)Ac, Be, (const CT *)Bc, Ce, (CT *)Cc);
  });
}

void launch_accumulate(int64_t n, int64_t nb, const int32_t *slice_e, const void *slice_c, const int32_t *off_e, const void *off_c,
                       int32_t *acc_e, void *acc_c, int first, int ring, cudaStream_t st) {
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    accumulate_kernel<R><<<grid_for(n, 256), 256, 0, st>>>(n, nb, slice_e, (const CT *)slice_c, off_e, (const CT *)off_c, acc_e,
                                                           (CT *)acc_c, first);
  });
}

void launch_finalize(int kind, int64_t B, const int32_t *root_e, const void *root_c, int64_t root_stride,
                     const int32_t *off_e, const void *off_c, int32_t *energy, uint64_t *count,
                     uint32_t *count_mod, int ring, cudaStream_t st) {
  BBTN_RING_DISPATCH(ring, {
    using CT = typename R::T;
    finalize_kernel<R><<<grid_for(B, 128), 128, 0, st>>>(kind, B, root_e, (const CT *)root_c, root_stride, off_e,
                                                         (const CT *)off_c, energy, count, count_mod, ring);
  });
}

}  // namespace bbtn
