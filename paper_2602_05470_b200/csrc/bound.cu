// bound.cu -- K5: warp-level region bounds used for pruning (sm_100a).
//
// PAPER.md:65 "BBTN prunes infeasible or suboptimal sub-TNs by evaluating local energy
// contributions over a subset of variables R"; :67 global pruning against the incumbent.
// The exact bound formula lives in the paper's missing supplement; reading A15 fixes
// ours: an exact max over the free vertices of every (disjoint) region of the terms inside
// region u F, plus the best entry of every term no region covers, plus the fixed-fixed terms.
// One warp per (leaf, region): the lanes enumerate the 2^nf region configurations and the
// maximum is taken with a warp-wide integer reduction (REDUX).
#include "../../include/bbtn.h"
#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

constexpr int WARPS = 8;

__global__ void __launch_bounds__(WARPS * 32) region_max_kernel(BoundTables t, const uint8_t *__restrict__ assign,
                                                                int64_t B, int32_t *__restrict__ scratch) {
  __shared__ int32_t sh_u[WARPS][32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t total = B * t.n_regions;
  for (int64_t item = blockIdx.x * (int64_t)WARPS + w; item < total; item += (int64_t)gridDim.x * WARPS) {
    const int64_t b = item / t.n_regions;
    const int j = (int)(item - b * t.n_regions);
    const int v0 = t.reg_off[j], nf = t.reg_off[j + 1] - v0;
    const uint8_t *x = assign + b * t.n_fixed;
    // per-bit unary coefficient: vertex term + terms to fixed neighbours.  MIS: forbid mask instead.
    int32_t u = lane < nf ? t.reg_vw[v0 + lane] : 0;
    uint32_t forbid = 0;
    for (int i = t.reg_fix_off[j]; i < t.reg_fix_off[j + 1]; i++) {
      const int bit = t.reg_fix_bit[i], xv = x[t.reg_fix_col[i]];
      if (t.kind == 0) { if (bit == lane) u += t.reg_fix_w[i] * (2 * xv - 1); }
      else if (xv) forbid |= 1u << bit;
    }
    __syncwarp();
    sh_u[w][lane] = u;
    __syncwarp();
    const int p0 = t.reg_pair_off[j], p1 = t.reg_pair_off[j + 1];
    int32_t best = NEG_INF;
    for (uint32_t cfg = lane; cfg < (1u << nf); cfg += 32) {
      int32_t s = 0; bool ok = true;
      if (t.kind == 0) {
        for (int q = 0; q < nf; q++) s += ((cfg >> q) & 1u) ? sh_u[w][q] : -sh_u[w][q];
        for (int i = p0; i < p1; i++) {
          const uint32_t d = ((cfg >> t.reg_pair_a[i]) ^ (cfg >> t.reg_pair_b[i])) & 1u;
          s += d ? -t.reg_pair_w[i] : t.reg_pair_w[i];
        }
      } else {
        ok = (cfg & forbid) == 0;
        for (int q = 0; q < nf; q++) if ((cfg >> q) & 1u) s += sh_u[w][q];
        for (int i = p0; i < p1 && ok; i++)
          if (((cfg >> t.reg_pair_a[i]) & (cfg >> t.reg_pair_b[i])) & 1u) ok = false;
      }
      if (ok && s > best) best = s;
    }
    best = __reduce_max_sync(0xffffffffu, best);
    if (lane == 0) scratch[item] = best;
    __syncwarp();
  }
}

__global__ void bound_sum_kernel(BoundTables t, const uint8_t *__restrict__ assign, int64_t B,
                                 const int32_t *__restrict__ scratch, int32_t *__restrict__ bound) {
  for (int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; b < B; b += (int64_t)gridDim.x * blockDim.x) {
    const uint8_t *x = assign + b * t.n_fixed;
    int64_t s = t.const_term; bool ok = true;
    for (int i = 0; i < t.n_ff; i++) {
      const int xu = x[t.ff_cu[i]], xv = x[t.ff_cv[i]];
      if (t.kind == 0) s += t.ff_w[i] * (2 * xu - 1) * (2 * xv - 1);
      else if (xu & xv) ok = false;
    }
    for (int i = 0; i < t.n_fv; i++) {
      const int xv = x[t.fv_c[i]];
      s += t.kind == 0 ? t.fv_w[i] * (2 * xv - 1) : (xv ? t.fv_w[i] : 0);
    }
    for (int i = 0; i < t.n_uv; i++) {          // MIS: free uncovered vertex may join unless a fixed neighbour is in
      bool allow = true;
      for (int q = t.uv_off[i]; q < t.uv_off[i + 1]; q++) if (x[t.uv_cols[q]]) allow = false;
      if (allow && t.uv_w[i] > 0) s += t.uv_w[i];
    }
    for (int j = 0; j < t.n_regions; j++) s += scratch[b * t.n_regions + j];
    // reported units: Ising lower bound on min H, MIS upper bound on the weight
    bound[b] = !ok ? NEG_INF : (t.kind == 0 ? (int32_t)(-s) : (int32_t)s);
  }
}

}  // namespace

void launch_region_bound(const BoundTables &t, const uint8_t *d_assign, int64_t B, int32_t *region_scratch,
                         int32_t *bound, cudaStream_t st) {
  if (t.n_regions > 0) {
    const int64_t items = B * t.n_regions;
    int64_t g = (items + WARPS - 1) / WARPS;
    if (g > 148 * 8) g = 148 * 8;
    region_max_kernel<<<(unsigned)g, WARPS * 32, 0, st>>>(t, d_assign, B, region_scratch);
  }
  int64_t g = (B + 127) / 128;
  if (g > 148 * 8) g = 148 * 8;
  bound_sum_kernel<<<(unsigned)g, 128, 0, st>>>(t, d_assign, B, region_scratch, bound);
}

// ---- the no-allocation variant (include/bbtn.h: bbtn_region_bound_static) ----------------------------------------
// The per-(leaf, region) maxima go to a file-scope device array instead of a buffer the handle allocates.  Every GPU
// that loads the library holds these 4 MiB until the process exits.  Every call shares the array and finds the last
// call's contents in it: region_max_kernel writes all B * n_regions entries before bound_sum_kernel reads them (same
// stream), so nothing needs clearing -- but two calls that overlap on the GPU (different streams) race on it.
static __device__ __align__(256) int32_t g_region_scratch[BBTN_REGION_BOUND_STATIC_MAX_ITEMS];

// In host code the name g_region_scratch is a stand-in, not a device address: ask the runtime, once per device, with
// that device current.
int launch_region_bound_static(const BoundTables &t, const uint8_t *d_assign, int64_t B, int32_t *bound, cudaStream_t st,
                               cudaError_t *cuda_err) {
  constexpr int MAX_DEV = 64;
  static int32_t *addr[MAX_DEV] = {};
  *cuda_err = cudaSuccess;
  int dev = -1;
  if ((*cuda_err = cudaGetDevice(&dev)) != cudaSuccess) return 1;
  if (dev < 0 || dev >= MAX_DEV) return 2;
  if (!addr[dev]) {
    int32_t *ptr = nullptr;
    if ((*cuda_err = cudaGetSymbolAddress((void **)&ptr, g_region_scratch)) != cudaSuccess || !ptr) return 1;
    addr[dev] = ptr;
  }
  if (B > 0) launch_region_bound(t, d_assign, B, addr[dev], bound, st);      // B = 0: set-up only
  return 0;
}

}  // namespace bbtn
