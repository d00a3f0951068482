// construct.cuh -- the entries of the input tensors (K1), shared by the construct kernels (kernels.cu) and the
// one-CTA-per-leaf tree kernel (fused_tree.cu).
#pragma once
#include "plan.h"
#include "ring.cuh"

namespace bbtn {

// ---------------------------------------------------------------------------------------------
// Input tensor entries, max-plus form (PAPER.md:49 Ising B and w, :55 MWIS B and w; A1-A3):
//   Ising  bond [su][sv] = +J*sigma(su)*sigma(sv), vertex [s] = +h*sigma(s), sigma(s) = 2s-1, count 1
//   MIS    bond = (0,1) except [1][1] = zero element; vertex = (0,1), (w,1)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int32_t entry_energy(int kind, int type, int32_t w, int su, int sv) {
  if (kind == 0) {
    int32_t s = (2 * su - 1) * (type == 0 ? (2 * sv - 1) : 1);
    return w * s;
  }
  if (type == 0) return (su & sv) ? NEG_INF : 0;
  return su ? w : 0;
}

// value of input tensor `r` at free bits (xu, xv), pre-summing single-owner indices (reading A7)
template <class R>
__device__ __forceinline__ void input_element(int kind, const InputRec &r, int fu_val, int fv_val, int xu, int xv,
                                              int32_t &e, typename R::T &c) {
  e = NEG_INF; c = czero<R>();
  const int nu = r.su ? 2 : 1, nv = r.sv ? 2 : 1;
  for (int a = 0; a < nu; a++)
    for (int b = 0; b < nv; b++) {
      int su = r.fu >= 0 ? fu_val : (r.su ? a : xu);
      int sv = r.v < 0 ? 0 : (r.fv >= 0 ? fv_val : (r.sv ? b : xv));
      int32_t ee = entry_energy(kind, r.type, r.w, su, sv);
      if (ee > ZERO_BELOW) oplus<R>(e, c, ee, R::from_small(1));
    }
}

}  // namespace bbtn
