// fused_tree.cu -- K1..K4 of a SMALL network in one launch: one CTA per leaf, every tensor in shared memory.
//
// Networks whose largest intermediate has a few thousand elements (BASELINE configs 1 and 2: 6x6 +-J lattice,
// width 6; King's subgraph 12x12, width 12-13) take hundreds of pairwise contractions (Eq. 2 evaluated pairwise,
// PAPER.md:51, :57) of a few hundred elements each: as separate launches, even inside a CUDA graph, they cost
// ~2 us of latency per tree node and do nothing else.  Here the CTA builds the sliced input tensors of its leaf
// (K1), walks the plan's steps in order -- C[o] = (+)_k A[fa(o) + ka(k)] (.) B[fb(o) + kb(k)], the streaming
// form of K3 with the bit permutations folded into the addressing -- with a block barrier between steps, and
// finalises (K4).  Leaf-invariant subtrees are recomputed by every CTA (cheaper than a second launch at this size).
// Step descriptors are prefetched two steps ahead (global -> register -> shared memory).
#include "construct.cuh"
#include "kernels.h"

namespace bbtn {
namespace {

// threads per CTA = 2^FTB: 256 in general; 128 for the smallest networks (every tensor <= 2^8 elements), where the
// block barrier between steps is most of a step's time

template <class R, int FTB>
__global__ void __launch_bounds__(1 << FTB, 1) fused_tree_kernel(int kind, const InputRec *__restrict__ inputs,
                                                           const int32_t *__restrict__ list_build, int n_build,
                                                           const int32_t *__restrict__ list_scalar, int n_scalar,
                                                           const uint8_t *__restrict__ assign, int n_fixed,
                                                           const FusedStep *__restrict__ steps, int n_steps,
                                                           int arena_elems, int inv_base, int result_off,
                                                           int32_t *__restrict__ energy, uint64_t *__restrict__ count,
                                                           uint32_t *__restrict__ count_mod, int ring, const FusedGlobal g,
                                                           int64_t Bn) {
  using CT = typename R::T;
  constexpr int FT = 1 << FTB;
  extern __shared__ __align__(16) unsigned char smem[];
  FusedStep *desc = reinterpret_cast<FusedStep *>(smem);                          // two descriptors, double-buffered
  int32_t *te = reinterpret_cast<int32_t *>(smem + 2 * sizeof(FusedStep));
  CT *tc = reinterpret_cast<CT *>(smem + 2 * sizeof(FusedStep) + (((size_t)arena_elems * 4 + 15) & ~(size_t)15));
  __shared__ int32_t off_e_s;
  __shared__ unsigned long long off_c_bits;
  const int64_t b = blockIdx.x;
  const uint8_t *asg = assign + b * n_fixed;
  const int t = threadIdx.x;
  constexpr int WORDS = (int)(sizeof(FusedStep) / 4);

  // descriptors travel global -> register -> shared memory TWO steps ahead: the word of step s+2 is requested while
  // step s runs and is parked in shared memory at the top of step s+1, so no step ever waits for a global load
  auto fetch = [&](int s) -> uint32_t {
    return (s < n_steps && t < WORDS) ? __ldg(reinterpret_cast<const uint32_t *>(steps + s) + t) : 0u;
  };
  auto park = [&](int s, uint32_t w) {               // descriptor word of step s -> desc[s & 1]
    if (s < n_steps && t < WORDS) reinterpret_cast<uint32_t *>(desc + (s & 1))[t] = w;
  };
  park(0, fetch(0));
  uint32_t pre = fetch(1);

  // ---- K1: the sliced input tensors of this leaf, and the product of its scalar inputs
  for (int i = t; i < n_build; i += FT) {
    const InputRec r = inputs[list_build[i]];
    const int fu_val = r.fu >= 0 ? asg[r.fu] : 0, fv_val = r.fv >= 0 ? asg[r.fv] : 0;
    const int base = g.build_off ? g.build_off[i] : (r.variant ? 0 : inv_base) + (int)r.offset;
    for (int x = 0; x < (1 << r.rank); x++) {
      int32_t e; CT c;
      input_element<R>(kind, r, fu_val, fv_val, r.bu >= 0 ? (x >> r.bu) & 1 : 0, r.bv >= 0 ? (x >> r.bv) & 1 : 0, e, c);
      te[base + x] = e; stc<R>(tc, base + x, c);
    }
  }
  if (t == 0 && g.finalize) {
    int32_t acc_e = 0; CT acc_c = R::from_small(1);
    for (int i = 0; i < n_scalar; i++) {
      const InputRec r = inputs[list_scalar[i]];
      int32_t e; CT c;
      input_element<R>(kind, r, r.fu >= 0 ? asg[r.fu] : 0, r.fv >= 0 ? asg[r.fv] : 0, 0, 0, e, c);
      acc_e += e; acc_c = R::mul(acc_c, c);
      canonicalise<R>(acc_e, acc_c);
    }
    off_e_s = acc_e;
    if constexpr (R::kCounts) off_c_bits = (unsigned long long)acc_c;
  }
  __syncthreads();

  // ---- K3, step by step
  for (int s = 0; s < n_steps; s++) {
    const FusedStep &d = desc[s & 1];
    park(s + 1, pre);
    pre = fetch(s + 2);
    const int rO = d.rO, nK = d.nK;
    const int32_t *ae = te + d.offA, *be = te + d.offB;
    const CT *ac = tc + d.offA, *bc = tc + d.offB;
    // a thread's outputs are o = t + j * FT: the low log2(FT) bits of o never change, their address part is computed once
    // (unused table entries are 0, so the loops below need no rank tests and unroll into independent loads)
    uint32_t a_lo = 0, b_lo = 0;
#pragma unroll
    for (int q = 0; q < FTB; q++) { const uint32_t m = 0u - ((t >> q) & 1u); a_lo += d.addA[q] & m; b_lo += d.addB[q] & m; }
    for (int o = t; o < (1 << rO); o += FT) {
      uint32_t a0 = a_lo, b0 = b_lo;
#pragma unroll
      for (int q = FTB; q < 13; q++) { const uint32_t m = 0u - ((o >> q) & 1u); a0 += d.addA[q] & m; b0 += d.addB[q] & m; }
      int32_t acc_e = NEG_INF; CT acc_c = czero<R>();
      if (nK <= 3) {
#pragma unroll 4
        for (int k = 0; k < (1 << nK); k++) {
          const uint32_t ia = a0 + d.kkA[k], ib = b0 + d.kkB[k];
          oplus<R>(acc_e, acc_c, ae[ia] + be[ib], R::mul(ldc<R>(ac, ia), ldc<R>(bc, ib)));
        }
      } else {
        for (int k = 0; k < (1 << nK); k++) {
          uint32_t ia = a0, ib = b0;
          for (int j = 0; j < nK; j++) if ((k >> j) & 1) { ia += d.kA[j]; ib += d.kB[j]; }
          oplus<R>(acc_e, acc_c, ae[ia] + be[ib], R::mul(ldc<R>(ac, ia), ldc<R>(bc, ib)));
        }
      }
      canonicalise<R>(acc_e, acc_c);
      te[d.offC + o] = acc_e; stc<R>(tc, d.offC + o, acc_c);
      if (d.gout >= 0) {                                 // a tensor the rest of the tree reads from the global arena
        const bool var = d.gout & 1;
        const int64_t gi = var ? (d.gout >> 1) * Bn + (b << rO) + o : (d.gout >> 1) + o;
        (var ? g.ve : g.ie)[gi] = acc_e;
        stc<R>(reinterpret_cast<CT *>(var ? g.vc : g.ic), gi, acc_c);
      }
    }
    __syncthreads();
  }
  if (!g.finalize) return;

  // ---- K4: offset (.) root, canonical, reported units
  if (t == 0) {
    int32_t e = off_e_s; CT c;
    if constexpr (R::kCounts) c = (CT)off_c_bits; else c = CT{};
    if (result_off >= 0) { e += te[result_off]; c = R::mul(c, ldc<R>(tc, result_off)); }
    canonicalise<R>(e, c);
    const bool zero = e == NEG_INF;
    if constexpr (!R::kCounts) {
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

}  // namespace

size_t fused_tree_smem_bytes(int arena_elems, int ring) {
  const size_t csz = ring_count_bytes(ring);
  return 2 * sizeof(FusedStep) + (((size_t)arena_elems * 4 + 15) & ~(size_t)15) + (size_t)arena_elems * csz + 16;
}

// Opt in to the device's maximum dynamic shared memory for the instantiation (ring, max_rank) will launch.  Call it
// outside any stream capture, before launch_fused_tree.
void configure_fused_tree(int ring, int max_rank) {
  int dev = 0, max_smem = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  max_smem -= 1024;                                        // the kernel's static shared memory counts against the same limit
  BBTN_RING_DISPATCH(ring, {
    if (max_rank <= 8) cudaFuncSetAttribute(fused_tree_kernel<R, 7>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    else cudaFuncSetAttribute(fused_tree_kernel<R, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
  });
}

void launch_fused_tree(int kind, const InputRec *d_inputs, const int32_t *d_list_build, int n_build,
                       const int32_t *d_list_scalar, int n_scalar, const uint8_t *d_assign, int n_fixed, int64_t B,
                       const FusedStep *d_steps, int n_steps, int arena_elems, int inv_base, int result_off,
                       int32_t *energy, uint64_t *count, uint32_t *count_mod, int ring, int max_rank, cudaStream_t st,
                       const FusedGlobal &g) {
  const size_t smem = fused_tree_smem_bytes(arena_elems, ring);
  BBTN_RING_DISPATCH(ring, {
    if (max_rank <= 8) {
      fused_tree_kernel<R, 7><<<(unsigned)B, 128, smem, st>>>(kind, d_inputs, d_list_build, n_build, d_list_scalar, n_scalar, d_assign,
                                                              n_fixed, d_steps, n_steps, arena_elems, inv_base, result_off, energy,
                                                              count, count_mod, ring, g, B);
    } else {
      fused_tree_kernel<R, 8><<<(unsigned)B, 256, smem, st>>>(kind, d_inputs, d_list_build, n_build, d_list_scalar, n_scalar, d_assign,
                                                              n_fixed, d_steps, n_steps, arena_elems, inv_base, result_off, energy,
                                                              count, count_mod, ring, g, B);
    }
  });
}

}  // namespace bbtn
