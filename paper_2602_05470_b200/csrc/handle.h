// handle.h -- private definition of bbtn_handle and shared host helpers (not part of the ABI).
#pragma once
#include <cuda_runtime.h>

#include <map>
#include <memory>
#include <string>
#include <vector>

#include "../../include/bbtn.h"
#include "kernels.h"
#include "plan.h"

namespace bbtn {

struct DevBuf {
  void *p = nullptr; size_t bytes = 0;
  DevBuf() = default;
  DevBuf(const DevBuf &) = delete;
  DevBuf &operator=(const DevBuf &) = delete;
  ~DevBuf() { if (p) cudaFree(p); }
  cudaError_t ensure(size_t n) {
    if (n <= bytes && p) return cudaSuccess;
    if (p) { cudaFree(p); p = nullptr; bytes = 0; }
    cudaError_t e = cudaMalloc(&p, n ? n : 1);
    if (e == cudaSuccess) bytes = n;
    return e;
  }
  template <class T> cudaError_t upload(const std::vector<T> &v) {
    cudaError_t e = ensure(v.size() * sizeof(T));
    if (e != cudaSuccess || v.empty()) return e;
    return cudaMemcpy(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
  }
};

struct DevPlan {
  Plan plan;
  DevBuf inputs, list_var, list_inv, list_scalar;
  int n_var = 0, n_inv = 0, n_scalar = 0;
  DevBuf var_e, var_c, inv_e, inv_c, off_e, off_c;
  DevBuf assign, energy, count, count_mod;      // staging for host-pointer calls
  // small networks (every tensor of a leaf fits shared memory): the whole plan runs as one launch (fused_tree.cu)
  DevBuf fused_steps, list_build;
  int fused = -1;                               // -1 not decided yet, 0 no, 1 yes
  int n_build = 0, fused_arena = 0;
  // larger networks: the SMALL SUBTREES of the plan (every tensor <= 2^hyb_rank elements) run as a shared-memory prologue,
  // one CTA per leaf (group 1: subtrees that end in a leaf-dependent tensor) or one CTA (group 0: leaf-invariant ones),
  // and only the rest of the tree as per-node launches (api.cu prepare_hybrid)
  int hybrid = -1;                              // -1 not decided yet, 0 no, 1 yes
  struct HybridGroup {
    std::vector<FusedStep> steps; std::vector<int32_t> build, build_off;
    int arena = 0, max_rank = 0;
    DevBuf d_steps, d_build, d_build_off;
  } hyb[2];
  std::vector<Step> hyb_big;                    // the steps that stay per-node launches, operands re-pointed at the prologue's outputs
  int hyb_rank = 0;
  int64_t hyb_max_B = 0;                        // the prologue pays while its CTAs fit about two waves; beyond, node-by-node launches batch better
  bool tables_ready = false;
  int64_t B_cap = 0;
  std::vector<cudaGraphExec_t> graphs;          // per ring, for graph_B
  int64_t graph_B = -1;
  const void *graph_io[4] = {nullptr, nullptr, nullptr, nullptr};
  ~DevPlan() { for (auto g : graphs) if (g) cudaGraphExecDestroy(g); }
};

struct BoundPlan {
  DevBuf tab[20];
  BoundTables t;
  DevBuf scratch, assign, bound;
};

int fail(bbtn_handle *h, int code, const std::string &msg);
bool have_device();
int run_plan(bbtn_handle *h, DevPlan *dp, const uint8_t *assign, int64_t B, int32_t *energy, uint64_t *count,
             uint32_t *count_mod, bool allow_graph, void *stream);

}  // namespace bbtn

struct bbtn_handle {
  bbtn::Problem P;
  std::string err;
  int force_mode = 0;
  std::map<std::vector<int32_t>, std::unique_ptr<bbtn::DevPlan>> plans;
  std::map<std::vector<int32_t>, std::unique_ptr<bbtn::BoundPlan>> bounds;
  // branching driver (branching.cu): the unsliced tree every leaf is planned on, and one scratch plan whose
  // device buffers are reused by every leaf (leaves have different fixed sets, so they are not cached)
  std::vector<std::vector<int>> sweep_orders;        // caller's base orders for the library's tree search (bbtn_add_sweep_order)
  // the plan bbtn_local_plan_query / bbtn_solve_local chose last (tree search over many candidates: not repeated for the same request)
  struct LocalChoice { int32_t log2_target = 0; int64_t budget = 0; size_t n_hints = 0; bbtn::LocalPlan lp; std::shared_ptr<bbtn::Problem> P; };
  std::unique_ptr<LocalChoice> local_choice;
  std::unique_ptr<bbtn::Problem> Pbr;
  std::unique_ptr<bbtn::DevPlan> scratch;
};

#define CUDA_TRY(h, expr)                                                                       \
  do {                                                                                          \
    cudaError_t _e = (expr);                                                                    \
    if (_e != cudaSuccess)                                                                      \
      return ::bbtn::fail(h, _e == cudaErrorMemoryAllocation ? BBTN_ENOMEM : BBTN_ECUDA,        \
                          std::string(#expr) + ": " + cudaGetErrorString(_e));                  \
  } while (0)
