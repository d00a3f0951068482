// kernels.h -- launchers of the sm_100a kernels (K1..K5).  All pointers are DEVICE pointers.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "plan.h"

namespace bbtn {

// counts mod 2^64 / no counts (search mode) / mod 2^31-1 and mod 2^31-19 packed in one 64-bit word (CRT mode's second pass)
enum RingId : int { RING_U64 = 0, RING_NONE = 3, RING_P12 = 4 };
inline size_t ring_count_bytes(int ring) { return ring == RING_NONE ? 0 : 8; }

constexpr int32_t kNegInf = -(1 << 30);
constexpr int32_t kZeroThreshold = -(1 << 29);   // e < threshold  <=>  zero element (reading A8)

// K1: build the sliced input tensors of every leaf and the per-leaf scalar offset.
//   d_inputs: InputRec table; d_list: ids to build (rank > 0); variant inputs are written for
//   b = 0..B-1 at arena offset off*B + b*2^rank, invariant ones once.
void launch_construct(int kind, const InputRec *d_inputs, const int32_t *d_list_var, int n_var,
                      const int32_t *d_list_inv, int n_inv, const int32_t *d_list_scalar, int n_scalar,
                      const uint8_t *d_assign, int n_fixed, int64_t B,
                      int32_t *var_e, void *var_c, int32_t *inv_e, void *inv_c,
                      int32_t *off_e, void *off_c, int ring, cudaStream_t st);

// K2: dst[b][pi(i)] = src[b][i], bit j of pi(i) = bit perm[j] of i.
void launch_permute(int rank, const int32_t *perm, int64_t batch, const int32_t *src_e, const void *src_c,
                    int32_t *dst_e, void *dst_c, int ring, cudaStream_t st);

// K3 (streaming form, permutation fused into the operand addressing) and its long-reduction form.
//   xs (local slicing, Step::n_slice > 0): device rows [nb][n_slice] of 0/1; an operand that is a view of a stored tensor
//   (Step::xA / xB) starts, for batch entry b, at its base + sum_j xs[b][j] * sliceA/B[j] instead of base + b * stride.
void launch_absorb(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                   int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs = nullptr);
bool launch_absorb_vec(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                       int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs = nullptr);
// the same with the tile's footprint of a mid-sized B staged in shared memory (absorb_stage.cu)
bool launch_absorb_stage(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                       int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs = nullptr);   // false: shape not covered, use launch_absorb's scalar kernel
void launch_reduce(const Step &s, int64_t nb, const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc,
                   int32_t *Ce, void *Cc, int ring, cudaStream_t st, const uint8_t *xs = nullptr);

// K3 (register/shared-memory tiled form).  C[b,g,m,n] = (+)_k A (.) B.
//   a_kmajor = 1: A is [g][k][m] (m fastest, the engine's canonical order); 0: A is row-major [m][k].
//   B is [g][k][n], C is [g][m][n].  Batch strides in elements (0 = shared).  count_bits <= 32 selects the
//   32-bit-operand multiply path, energy_bits <= 11 (with 32-bit accumulators) the packed 16x2 form (RING_U64 only).
void launch_gemm_tiled(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                       const int32_t *Ae, const void *Ac, const int32_t *Be, const void *Bc, int32_t *Ce, void *Cc,
                       int64_t sA, int64_t sB, int64_t sC, int ring, int count_bits, int energy_bits, cudaStream_t st);

// K3 v2 for the mod-2^64 ring (gemm_tiled.cu): chunked two-pass kernel, 4 integer instructions per FMA.
void launch_gemm_tiled_u64(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                           const int32_t *Ae, const uint64_t *Ac, const int32_t *Be, const uint64_t *Bc,
                           int32_t *Ce, uint64_t *Cc, int64_t sA, int64_t sB, int64_t sC, int count_bits, int energy_bits,
                           cudaStream_t st);

bool gemm_pack16_eligible(int K, int count_bits, int energy_bits);

// K3 packed form (gemm_pack16.cu; 128 x 128 tile, 64 x 64 for M, N <= 64): two outputs per integer instruction; finite |energy| < 2^11, 32-bit accumulators.
void launch_gemm_pack16(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor,
                        const int32_t *Ae, const uint64_t *Ac, const int32_t *Be, const uint64_t *Bc,
                        int32_t *Ce, uint64_t *Cc, int64_t sA, int64_t sB, int64_t sC, int count_bits, cudaStream_t st);

// K3 in search mode (gemm_maxplus.cu): max-plus on the energy planes alone, one fused add-max per FMA (two with
// energy_bits <= 11: packed 16-bit halves); layout arguments as launch_gemm_tiled.
void launch_gemm_maxplus(int64_t batch, int64_t G, int M, int N, int K, int a_kmajor, const int32_t *A, const int32_t *B,
                         int32_t *C, int64_t sA, int64_t sB, int64_t sC, int energy_bits, cudaStream_t st);

// Local slicing: acc (+)= (+)_b offset[b] (.) slice[b], element-wise over n elements, nb slices stored [nb][n]
// (first = 1: acc is overwritten); the zero tensor when slice_e == nullptr.  offset[b] is one element per slice on the
// device.  (+) over the assignments of a segment's locally fixed indices (Eq. 3, on a sub-network).
void launch_accumulate(int64_t n, int64_t nb, const int32_t *slice_e, const void *slice_c, const int32_t *off_e, const void *off_c,
                       int32_t *acc_e, void *acc_c, int first, int ring, cudaStream_t st);

// K1..K4 of a small network in ONE launch (fused_tree.cu): one CTA per leaf, every tensor in shared memory.
// A step is C[o] = (+)_k A[fa(o) + ka(k)] (.) B[fb(o) + kb(k)] with shared-memory element offsets.
struct FusedStep {
  int32_t rO, nK, offA, offB, offC, pad;
  uint16_t addA[16], addB[16], kA[16], kB[16];   // unused entries are 0
  uint16_t kkA[8], kkB[8];                        // nK <= 3: the summed offsets of every k, ready to add
  int64_t gout;                                   // -1, or (global element offset << 1) | variant: the output also goes to the arena
};
// The same kernel as a PROLOGUE of a larger plan (api.cu prepare_hybrid): it contracts the small subtrees of every
// leaf in shared memory and writes the tensor each of them ends in to the global arena, where the per-node launches
// of the rest of the tree pick it up.  build_off != nullptr: shared-memory offsets of the inputs to build (parallel
// to list_build); steps with gout >= 0 store their output at ve + off * B + b * 2^rO (variant) or ie + off; finalize = 0.
struct FusedGlobal {
  const int32_t *build_off = nullptr;
  int32_t *ve = nullptr; void *vc = nullptr; int32_t *ie = nullptr; void *ic = nullptr;
  int finalize = 1;
};
size_t fused_tree_smem_bytes(int arena_elems, int ring);
void configure_fused_tree(int ring, int max_rank);     // outside stream capture, before the first launch of that instantiation
void launch_fused_tree(int kind, const InputRec *d_inputs, const int32_t *d_list_build, int n_build,
                       const int32_t *d_list_scalar, int n_scalar, const uint8_t *d_assign, int n_fixed, int64_t B,
                       const FusedStep *d_steps, int n_steps, int arena_elems, int inv_base, int result_off,
                       int32_t *energy, uint64_t *count, uint32_t *count_mod, int ring, int max_rank, cudaStream_t st,
                       const FusedGlobal &g = FusedGlobal());

// K4: (E[b], c[b]) = offset[b] (.) root[b]; canonicalise; convert to reported units.
//   root_e == nullptr: the network is all scalars.  root_stride 0: root is leaf-invariant.
void launch_finalize(int kind, int64_t B, const int32_t *root_e, const void *root_c, int64_t root_stride,
                     const int32_t *off_e, const void *off_c, int32_t *energy, uint64_t *count,
                     uint32_t *count_mod, int ring, cudaStream_t st);

// K5: warp-level region bounds (reading A15).
struct BoundTables {                 // device CSR tables built once per (regions, F)
  int kind, n_regions, n_fixed;
  const int32_t *reg_off;            // [n_regions+1] free vertices of each region
  const int32_t *reg_vw;             // vertex weight of each free region vertex
  const int32_t *reg_fix_off;        // [n_regions+1] per-region unary terms from fixed neighbours
  const int32_t *reg_fix_bit, *reg_fix_col, *reg_fix_w;   // local bit, assign column, coupling
  const int32_t *reg_pair_off;       // [n_regions+1] bonds inside the region
  const int32_t *reg_pair_a, *reg_pair_b, *reg_pair_w;    // local bits, coupling
  // terms outside every region
  int n_ff; const int32_t *ff_cu, *ff_cv, *ff_w;          // fixed-fixed bonds: assign columns, coupling
  int n_fv; const int32_t *fv_c, *fv_w;                   // fixed vertices: column, weight
  int n_uf; const int32_t *uf_c, *uf_w;                   // uncovered bonds with one fixed endpoint: column, coupling
  int n_uv; const int32_t *uv_off, *uv_cols, *uv_w;       // MIS: uncovered free vertices: CSR of fixed-neighbour columns, weight
  int32_t const_term;                                     // assignment-independent part
};
void launch_region_bound(const BoundTables &t, const uint8_t *d_assign, int64_t B, int32_t *region_scratch,
                         int32_t *bound, cudaStream_t st);
// the same with the region scratch in a file-scope device array (bound.cu); 0 = launched, 1 = CUDA error (*cuda_err),
// 2 = device ordinal out of range
int launch_region_bound_static(const BoundTables &t, const uint8_t *d_assign, int64_t B, int32_t *bound, cudaStream_t st,
                               cudaError_t *cuda_err);

// register-only integer microbenchmarks (include/bbtn.h: bbtn_int32_microbench)
int run_microbench(int which, int iters, double *ms, double *ops, cudaStream_t st);

}  // namespace bbtn
