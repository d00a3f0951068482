// api.cu -- the C ABI of include/bbtn.h: handle, plan cache, device arena, launch sequencing.
// Host logic only; every arithmetic step of the path runs in the kernels (kernels.h).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <string>
#include <vector>

#include "handle.h"

using namespace bbtn;

namespace bbtn {
thread_local std::string g_err;
int fail(bbtn_handle *h, int code, const std::string &msg) {
  if (h) h->err = msg;
  g_err = msg;
  return code;
}
bool have_device() {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return false; }
  return true;
}
}  // namespace bbtn

namespace {

// ---- debug checks of the raw-GEMM promises (include/bbtn.h: bbtn_set_debug_checks) ----
bool g_debug_checks = [] { const char *e = std::getenv("BBTN_DEBUG_CHECKS"); return e && e[0] == '1'; }();

// flags |= 1: a count >= 2^count_bits;  |= 2: an energy that is neither BBTN_NEG_INF nor within +-BBTN_ENERGY_LIMIT
__global__ void check_operand_kernel(const int32_t *__restrict__ e, const uint64_t *__restrict__ c, int64_t rows, int64_t row_len,
                                     int64_t row_stride, int count_bits, int energy_limit, int *flags) {
  const int64_t total = rows * row_len;
  int bad = 0;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = t / row_len, i = r * row_stride + (t - r * row_len);
    const int32_t ee = e[i];
    if (count_bits < 64 && c && (c[i] >> count_bits) != 0) bad |= 1;
    if (ee != BBTN_NEG_INF && (ee > energy_limit || ee < -energy_limit)) bad |= 2;
  }
  if (bad) atomicOr(flags, bad);
}

int check_gemm_operands(int64_t batch, int32_t M, int32_t N, int32_t K, const int32_t *Ae, const uint64_t *Ac, const int32_t *Be,
                        const uint64_t *Bc, int64_t sA, int64_t sB, int32_t count_bits, int32_t energy_bits, cudaStream_t st) {
  int *d_flags = nullptr, h_flags = 0;
  CUDA_TRY(nullptr, cudaMalloc(&d_flags, sizeof(int)));
  cudaMemsetAsync(d_flags, 0, sizeof(int), st);
  const int lim = energy_bits >= 29 ? BBTN_ENERGY_LIMIT : (1 << energy_bits) - 1;
  check_operand_kernel<<<148 * 4, 256, 0, st>>>(Ae, Ac, sA ? batch : 1, (int64_t)M * K, sA, count_bits, lim, d_flags);
  check_operand_kernel<<<148 * 4, 256, 0, st>>>(Be, Bc, sB ? batch : 1, (int64_t)K * N, sB, count_bits, lim, d_flags);
  cudaError_t e = cudaMemcpyAsync(&h_flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_flags);
  CUDA_TRY(nullptr, e);
  if (h_flags & 1) return fail(nullptr, BBTN_EINVAL, "debug check: an operand count is not below 2^count_bits (count_bits = " + std::to_string(count_bits) + ")");
  if (h_flags & 2) return fail(nullptr, BBTN_EINVAL, "debug check: an operand energy is neither BBTN_NEG_INF nor below 2^energy_bits in magnitude (energy_bits = " + std::to_string(energy_bits) + ")");
  return BBTN_OK;
}

int check_gemm_shape(int64_t batch, int32_t M, int32_t N, int32_t count_bits, int32_t energy_bits) {
  if (count_bits < 1 || count_bits > 64) return fail(nullptr, BBTN_EINVAL, "count_bits must be in 1..64");
  if (energy_bits < 1 || energy_bits > 32) return fail(nullptr, BBTN_EINVAL, "energy_bits must be in 1..32");
  // the smallest tile any K3 form uses is 64x64: one thread block per tile and batch entry
  const double n_cta = (double)((M + 63) / 64) * (double)((N + 63) / 64) * (double)batch;
  if (n_cta > 2147483647.0) return fail(nullptr, BBTN_ESHAPE, "GEMM launch would need more than 2^31-1 thread blocks; split the batch");
  return BBTN_OK;
}

void prepare_hybrid(bbtn_handle *h, DevPlan *dp);

int get_plan(bbtn_handle *h, const int32_t *fixed, int32_t n_fixed, bool enforce, DevPlan **out) {
  if (n_fixed < 0 || (n_fixed > 0 && !fixed)) return fail(h, BBTN_EINVAL, "bad fixed set");
  std::vector<int32_t> key(fixed, fixed + n_fixed);
  auto it = h->plans.find(key);
  if (it == h->plans.end()) {
    auto dp = std::make_unique<DevPlan>();
    std::string err;
    int rc = make_plan(h->P, key, h->force_mode, false, dp->plan, err);
    if (rc) return fail(h, rc, err);
    prepare_hybrid(h, dp.get());
    it = h->plans.emplace(key, std::move(dp)).first;
  }
  DevPlan *dp = it->second.get();
  if (enforce && dp->plan.rho > 0)
    return fail(h, BBTN_ESHAPE, "an intermediate of rank " + std::to_string(dp->plan.max_rank) +
                                    " exceeds max_elements_per_leaf (Eq. 4 rho = " + std::to_string(dp->plan.rho) + ")");
  *out = dp;
  return BBTN_OK;
}

int upload_tables(bbtn_handle *h, DevPlan *dp) {
  if (dp->tables_ready) return BBTN_OK;
  const Plan &pl = dp->plan;
  std::vector<int32_t> lv, li;
  for (size_t t = 0; t < pl.inputs.size(); t++) {
    if (pl.inputs[t].rank == 0) continue;
    (pl.inputs[t].variant ? lv : li).push_back((int32_t)t);
  }
  dp->n_var = (int)lv.size(); dp->n_inv = (int)li.size(); dp->n_scalar = (int)pl.scalar_inputs.size();
  CUDA_TRY(h, dp->inputs.ensure(pl.inputs.size() * sizeof(InputRec)));
  CUDA_TRY(h, cudaMemcpy(dp->inputs.p, pl.inputs.data(), pl.inputs.size() * sizeof(InputRec), cudaMemcpyHostToDevice));
  CUDA_TRY(h, dp->list_var.ensure(lv.size() * 4));
  CUDA_TRY(h, dp->list_inv.ensure(li.size() * 4));
  CUDA_TRY(h, dp->list_scalar.ensure(pl.scalar_inputs.size() * 4));
  if (!lv.empty()) CUDA_TRY(h, cudaMemcpy(dp->list_var.p, lv.data(), lv.size() * 4, cudaMemcpyHostToDevice));
  if (!li.empty()) CUDA_TRY(h, cudaMemcpy(dp->list_inv.p, li.data(), li.size() * 4, cudaMemcpyHostToDevice));
  if (!pl.scalar_inputs.empty())
    CUDA_TRY(h, cudaMemcpy(dp->list_scalar.p, pl.scalar_inputs.data(), pl.scalar_inputs.size() * 4, cudaMemcpyHostToDevice));
  CUDA_TRY(h, dp->inv_e.ensure((size_t)pl.arena_invariant_elems * 4));
  CUDA_TRY(h, dp->inv_c.ensure((h->P.flags & BBTN_SEARCH_ONLY) ? 0 : (size_t)pl.arena_invariant_elems * 8));
  if (dp->hybrid == 1)
    for (auto &g : dp->hyb) {
      if (g.steps.empty()) continue;
      CUDA_TRY(h, g.d_steps.ensure(g.steps.size() * sizeof(FusedStep)));
      CUDA_TRY(h, cudaMemcpy(g.d_steps.p, g.steps.data(), g.steps.size() * sizeof(FusedStep), cudaMemcpyHostToDevice));
      CUDA_TRY(h, g.d_build.upload(g.build));
      CUDA_TRY(h, g.d_build_off.upload(g.build_off));
    }
  dp->tables_ready = true;
  return BBTN_OK;
}

// descriptor of one streaming step with shared-memory operand offsets (fused_tree.cu)
FusedStep make_fused_step(const Step &s, int64_t offA, int64_t offB, int64_t offC) {
  FusedStep f;
  std::memset(&f, 0, sizeof(f));
  f.rO = s.rO; f.nK = s.nK; f.gout = -1;
  f.offA = (int32_t)offA; f.offB = (int32_t)offB; f.offC = (int32_t)offC;
  for (int q = 0; q < s.rO; q++) { f.addA[q] = (uint16_t)s.addA[q]; f.addB[q] = (uint16_t)s.addB[q]; }
  for (int j = 0; j < s.nK; j++) { f.kA[j] = (uint16_t)s.kA[j]; f.kB[j] = (uint16_t)s.kB[j]; }
  if (s.nK <= 3)
    for (int k = 0; k < (1 << s.nK); k++)
      for (int j = 0; j < s.nK; j++) if ((k >> j) & 1) { f.kkA[k] += (uint16_t)s.kA[j]; f.kkB[k] += (uint16_t)s.kB[j]; }
  return f;
}

// Can the plan run as one launch with every tensor of a leaf in shared memory?  (fused_tree.cu)
int prepare_fused(bbtn_handle *h, DevPlan *dp) {
  if (dp->fused >= 0) return BBTN_OK;
  dp->fused = 0;
  const Plan &pl = dp->plan;
  if (h->P.flags & BBTN_NO_FUSED) return BBTN_OK;
  const int64_t arena = pl.arena_variant_elems + pl.arena_invariant_elems;
  if (pl.max_rank > 13 || arena > 60000 || pl.steps.empty()) return BBTN_OK;
  int max_smem = 0, dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if ((int64_t)fused_tree_smem_bytes((int)arena, RING_U64) > (int64_t)max_smem) return BBTN_OK;
  std::vector<FusedStep> fs;
  for (const Step &s : pl.steps) {
    if ((s.kind != STEP_ABSORB && s.kind != STEP_REDUCE) || s.rO > 13 || s.nK > 13 || s.n_slice) return BBTN_OK;
    fs.push_back(make_fused_step(s, (s.vA ? 0 : pl.arena_variant_elems) + s.offA, (s.vB ? 0 : pl.arena_variant_elems) + s.offB,
                                 (s.vC ? 0 : pl.arena_variant_elems) + s.offC));
  }
  std::vector<int32_t> lb;
  for (size_t t = 0; t < pl.inputs.size(); t++) if (pl.inputs[t].rank > 0) lb.push_back((int32_t)t);
  CUDA_TRY(h, dp->fused_steps.ensure(fs.size() * sizeof(FusedStep)));
  CUDA_TRY(h, cudaMemcpy(dp->fused_steps.p, fs.data(), fs.size() * sizeof(FusedStep), cudaMemcpyHostToDevice));
  CUDA_TRY(h, dp->list_build.upload(lb));
  dp->n_build = (int)lb.size(); dp->fused_arena = (int)arena;
  dp->fused = 1;
  return BBTN_OK;
}

// first-fit allocator over shared-memory element offsets (blocks are multiples of 4 elements)
struct SmallArena {
  std::map<int, int> free_; int top = 0;
  static int r4(int n) { return (n + 3) & ~3; }
  int alloc(int n) {
    n = r4(n);
    for (auto it = free_.begin(); it != free_.end(); ++it)
      if (it->second >= n) { const int off = it->first, rest = it->second - n; free_.erase(it); if (rest) free_[off + n] = rest; return off; }
    if (!free_.empty()) {
      auto last = std::prev(free_.end());
      if (last->first + last->second == top) { const int off = last->first; top = off + n; free_.erase(last); return off; }
    }
    const int off = top; top += n; return off;
  }
  void release(int off, int n) {
    n = r4(n);
    auto it = free_.emplace(off, n).first;
    auto nx = std::next(it);
    if (nx != free_.end() && it->first + it->second == nx->first) { it->second += nx->second; free_.erase(nx); }
    if (it != free_.begin()) { auto pv = std::prev(it); if (pv->first + pv->second == it->first) { pv->second += it->second; free_.erase(it); } }
  }
};

// Larger plans: most tree nodes are tiny (a few hundred elements) and, launched one by one, cost a few microseconds of
// latency each.  A node is SMALL if it is a streaming node and every tensor of its subtree has at most 2^R elements;
// the maximal small subtrees run in shared memory as a prologue (fused_tree.cu, one CTA per leaf for those that end in
// a leaf-dependent tensor, one CTA for the leaf-invariant ones) and write the tensor they end in to fresh storage
// behind the planned arenas (their planned slots may still be occupied that early); the remaining nodes keep their
// per-node launches with those operands re-pointed.  Host logic only; R is the largest of 12 .. 8 that fits.
void prepare_hybrid(bbtn_handle *h, DevPlan *dp) {
  if (dp->hybrid >= 0) return;
  dp->hybrid = 0;
  Plan &pl = dp->plan;
  if ((h->P.flags & BBTN_NO_FUSED) || pl.steps.size() < 48) return;
  if (pl.max_rank <= 13 && pl.arena_variant_elems + pl.arena_invariant_elems <= 60000 &&
      (int64_t)fused_tree_smem_bytes((int)(pl.arena_variant_elems + pl.arena_invariant_elems), RING_U64) <= 227 * 1024 - 1024)
    return;                                                // the one-launch form takes it (prepare_fused)
  const int n_in = (int)pl.inputs.size(), n_st = (int)pl.steps.size();
  std::map<std::pair<int, int64_t>, int> owner;              // (arena, offset) -> the tensor stored there right now
  for (int t = 0; t < n_in; t++) if (pl.inputs[t].rank > 0) owner[{pl.inputs[t].variant, pl.inputs[t].offset}] = t;
  std::vector<int> opA(n_st, -1), opB(n_st, -1), consumer(n_in + n_st, -1);
  for (int s = 0; s < n_st; s++) {
    const Step &st = pl.steps[s];
    if (st.n_slice || st.xA || st.xB) return;
    auto fa = owner.find({st.vA, st.offA});
    if (fa == owner.end()) return;
    opA[s] = fa->second; consumer[opA[s]] = s;
    if (st.kind != STEP_PERMUTE) {
      auto fb = owner.find({st.vB, st.offB});
      if (fb == owner.end()) return;
      opB[s] = fb->second; consumer[opB[s]] = s;
    }
    owner[{st.vC, st.offC}] = n_in + s;
  }
  const int64_t smem_cap = 227 * 1024 - 2048;
  for (int R = 12; R >= 8; R--) {
    std::vector<char> small(n_in + n_st, 0);
    for (int t = 0; t < n_in; t++) small[t] = pl.inputs[t].rank > 0 && pl.inputs[t].rank <= R;
    int n_small = 0; bool whole = false;
    for (int s = 0; s < n_st; s++) {
      const Step &st = pl.steps[s];
      small[n_in + s] = (st.kind == STEP_ABSORB || st.kind == STEP_REDUCE) && st.rO <= R && st.nK <= 13 && st.rA <= R && st.rB <= R &&
                        small[opA[s]] && opB[s] >= 0 && small[opB[s]];
      if (small[n_in + s]) { n_small++; if (consumer[n_in + s] < 0) whole = true; }
    }
    if (whole) return;                                       // the whole tree is small: the one-launch form takes it
    if (n_small < 24) return;
    // group of every small step = leaf dependence of the tensor its subtree ends in
    std::vector<int> grp(n_st, -1); std::vector<char> root(n_st, 0);
    for (int s = n_st - 1; s >= 0; s--) {
      if (!small[n_in + s]) continue;
      const int c = consumer[n_in + s];
      if (!small[n_in + c]) { root[s] = 1; grp[s] = pl.steps[s].vC ? 1 : 0; } else grp[s] = grp[c];
    }
    DevPlan::HybridGroup gnew[2];
    std::vector<int64_t> newoff(n_st, -1);
    int64_t ext[2] = {0, 0};
    bool fits = true;
    for (int g = 0; g < 2 && fits; g++) {
      SmallArena sm; std::map<int, int> loc;
      for (int s = 0; s < n_st; s++) {
        if (grp[s] != g) continue;
        for (int op : {opA[s], opB[s]})
          if (op < n_in && !loc.count(op)) { loc[op] = sm.alloc(1 << pl.inputs[op].rank); gnew[g].build.push_back(op); gnew[g].build_off.push_back(loc[op]); }
      }
      for (int s = 0; s < n_st; s++) {
        if (grp[s] != g) continue;
        const Step &st = pl.steps[s];
        const int offC = sm.alloc(1 << st.rO);
        FusedStep f = make_fused_step(st, loc[opA[s]], loc[opB[s]], offC);
        for (int op : {opA[s], opB[s]}) if (op >= n_in) sm.release(loc[op], 1 << pl.steps[op - n_in].rO);
        loc[n_in + s] = offC;
        if (root[s]) {
          const int64_t base = g ? pl.arena_variant_elems : pl.arena_invariant_elems;
          newoff[s] = base + ext[g];
          ext[g] += (((int64_t)1 << st.rO) + 3) & ~(int64_t)3;
          f.gout = (newoff[s] << 1) | g;
          sm.release(offC, 1 << st.rO);
        }
        gnew[g].steps.push_back(f);
        gnew[g].max_rank = std::max(gnew[g].max_rank, (int)st.rO);
      }
      gnew[g].arena = sm.top;
      if ((int64_t)fused_tree_smem_bytes(sm.top, RING_U64) > smem_cap) fits = false;
    }
    if (!fits) continue;
    for (int s = 0; s < n_st; s++) {
      if (small[n_in + s]) continue;
      Step st = pl.steps[s];
      if (opA[s] >= n_in && newoff[opA[s] - n_in] >= 0) st.offA = newoff[opA[s] - n_in];
      if (opB[s] >= n_in && newoff[opB[s] - n_in] >= 0) st.offB = newoff[opB[s] - n_in];
      dp->hyb_big.push_back(st);
    }
    for (int g = 0; g < 2; g++) { dp->hyb[g].steps = std::move(gnew[g].steps); dp->hyb[g].build = std::move(gnew[g].build);
                                  dp->hyb[g].build_off = std::move(gnew[g].build_off); dp->hyb[g].arena = gnew[g].arena; dp->hyb[g].max_rank = gnew[g].max_rank; }
    pl.arena_invariant_elems += ext[0]; pl.arena_variant_elems += ext[1];
    dp->hyb_rank = R;
    // One CTA per leaf walks hundreds of nodes at ~0.5 us each, so the prologue's time grows with the number of waves of
    // CTAs, while the per-node launches it replaces cost a few microseconds each whatever the batch: use it up to two waves
    // (measured on the 24x24 lattice: 256 leaves 18.0 -> 17.1 ms, 1024 leaves 20.4 -> 21.2 ms, 4096 leaves 34 -> 46 ms)
    const int64_t per_cta = (int64_t)fused_tree_smem_bytes(dp->hyb[1].arena, RING_U64) + 1024;
    dp->hyb_max_B = dp->hyb[1].steps.empty() ? INT64_MAX : 2 * 148 * std::max<int64_t>(1, (227 * 1024) / per_cta);
    dp->hybrid = 1;
    return;
  }
}

int ensure_batch(bbtn_handle *h, DevPlan *dp, int64_t B, bool host_io) {
  const Plan &pl = dp->plan;
  if (B > dp->B_cap && dp->fused != 1) {
    size_t need = (size_t)pl.arena_variant_elems * (size_t)B;
    size_t free_b = 0, total_b = 0;
    CUDA_TRY(h, cudaMemGetInfo(&free_b, &total_b));
    const size_t per_elem = (h->P.flags & BBTN_SEARCH_ONLY) ? 4 : 12;      // search mode has no count plane
    if (need * per_elem > free_b + dp->var_e.bytes + dp->var_c.bytes)
      return fail(h, BBTN_ENOMEM, "batch needs " + std::to_string(need * per_elem) + " bytes of device memory");
    CUDA_TRY(h, dp->var_e.ensure(need * 4));
    CUDA_TRY(h, dp->var_c.ensure(need * (per_elem - 4)));
    CUDA_TRY(h, dp->off_e.ensure((size_t)B * 4));
    CUDA_TRY(h, dp->off_c.ensure((size_t)B * 8));
    dp->B_cap = B;
  }
  if (host_io) {
    CUDA_TRY(h, dp->assign.ensure((size_t)B * std::max<size_t>(pl.fixed.size(), 1)));
    CUDA_TRY(h, dp->energy.ensure((size_t)B * 4));
    CUDA_TRY(h, dp->count.ensure((size_t)B * 8));
    CUDA_TRY(h, dp->count_mod.ensure((size_t)B * 8));
  }
  return BBTN_OK;
}

// enqueue the whole contraction for one count ring
void enqueue_ring(const bbtn_handle *h, DevPlan *dp, int64_t B, const uint8_t *d_assign, int32_t *d_energy,
                  uint64_t *d_count, uint32_t *d_count_mod, int ring, cudaStream_t st) {
  const Plan &pl = dp->plan;
  int32_t *ve = (int32_t *)dp->var_e.p, *ie = (int32_t *)dp->inv_e.p;
  char *vc = (char *)dp->var_c.p, *ic = (char *)dp->inv_c.p;
  const size_t csz = ring_count_bytes(ring);
  launch_construct(h->P.kind, (const InputRec *)dp->inputs.p, (const int32_t *)dp->list_var.p, dp->n_var,
                   (const int32_t *)dp->list_inv.p, dp->n_inv, (const int32_t *)dp->list_scalar.p, dp->n_scalar,
                   d_assign, (int)pl.fixed.size(), B, ve, vc, ie, ic, (int32_t *)dp->off_e.p, dp->off_c.p, ring, st);
  int energy_bits = 0;                                   // every finite energy of every tensor is within +-energy_range
  while (energy_bits < 32 && ((int64_t)1 << energy_bits) <= h->P.energy_range) energy_bits++;
  auto pe = [&](int v, int64_t off) { return v ? ve + off * B : ie + off; };
  auto pc = [&](int v, int64_t off) { return (void *)(v ? vc + (size_t)off * B * csz : ic + (size_t)off * csz); };
  const bool hyb = dp->hybrid == 1 && B <= dp->hyb_max_B;
  if (hyb)                                               // the small subtrees of every leaf, in shared memory (prepare_hybrid)
    for (int g = 0; g < 2; g++) {
      const DevPlan::HybridGroup &hg = dp->hyb[g];
      if (hg.steps.empty()) continue;
      FusedGlobal fg;
      fg.build_off = (const int32_t *)hg.d_build_off.p; fg.ve = ve; fg.vc = vc; fg.ie = ie; fg.ic = ic; fg.finalize = 0;
      launch_fused_tree(h->P.kind, (const InputRec *)dp->inputs.p, (const int32_t *)hg.d_build.p, (int)hg.build.size(), nullptr, 0,
                        d_assign, (int)pl.fixed.size(), g ? B : 1, (const FusedStep *)hg.d_steps.p, (int)hg.steps.size(), hg.arena, 0, -1,
                        nullptr, nullptr, nullptr, ring, hg.max_rank, st, fg);
    }
  for (const Step &s : hyb ? dp->hyb_big : pl.steps) {
    const int64_t nb = s.variant ? B : 1;
    switch (s.kind) {
      case STEP_ABSORB:
        launch_absorb(s, nb, pe(s.vA, s.offA), pc(s.vA, s.offA), pe(s.vB, s.offB), pc(s.vB, s.offB),
                      pe(s.vC, s.offC), pc(s.vC, s.offC), ring, st);
        break;
      case STEP_REDUCE:
        launch_reduce(s, nb, pe(s.vA, s.offA), pc(s.vA, s.offA), pe(s.vB, s.offB), pc(s.vB, s.offB),
                      pe(s.vC, s.offC), pc(s.vC, s.offC), ring, st);
        break;
      case STEP_PERMUTE:
        launch_permute(s.rO, s.perm, nb, pe(s.vA, s.offA), pc(s.vA, s.offA), pe(s.vC, s.offC), pc(s.vC, s.offC), ring, st);
        break;
      case STEP_GEMM:
        launch_gemm_tiled(nb, (int64_t)1 << s.lg, 1 << s.lm, 1 << s.ln, 1 << s.lk, 1,
                          pe(s.vA, s.offA), pc(s.vA, s.offA), pe(s.vB, s.offB), pc(s.vB, s.offB),
                          pe(s.vC, s.offC), pc(s.vC, s.offC),
                          s.vA ? ((int64_t)1 << s.rA) : 0, s.vB ? ((int64_t)1 << s.rB) : 0, (int64_t)1 << s.rO,
                          ring, s.count_bits, energy_bits, st);
        break;
    }
  }
  const bool has_root = pl.result_offset >= 0;
  launch_finalize(h->P.kind, B, has_root ? pe(pl.result_variant, pl.result_offset) : nullptr,
                  has_root ? pc(pl.result_variant, pl.result_offset) : nullptr, pl.result_variant ? 1 : 0,
                  (const int32_t *)dp->off_e.p, dp->off_c.p, d_energy, d_count, d_count_mod, ring, st);
}

}  // namespace

extern "C" {

const char *bbtn_version(void) { return "bbtn-b200 0.1 (sm_100a)"; }

const char *bbtn_last_error(const bbtn_handle *h) { return h ? h->err.c_str() : bbtn::g_err.c_str(); }

int bbtn_build(const bbtn_problem_desc *d, bbtn_handle **out) {
  if (!d || !out) return fail(nullptr, BBTN_EINVAL, "null argument");
  *out = nullptr;
  if (d->kind != BBTN_ISING && d->kind != BBTN_MIS) return fail(nullptr, BBTN_EINVAL, "unknown kind");
  if (d->n_vertices < 0 || d->n_edges < 0 || (d->n_edges > 0 && (!d->edge_u || !d->edge_v)))
    return fail(nullptr, BBTN_EINVAL, "bad graph");
  auto h = std::make_unique<bbtn_handle>();
  Problem &P = h->P;
  P.kind = d->kind; P.n = d->n_vertices; P.m = d->n_edges; P.flags = d->flags;
  P.eu.assign(d->edge_u, d->edge_u + P.m); P.ev.assign(d->edge_v, d->edge_v + P.m);
  std::vector<std::pair<int, int>> seen;
  int64_t range = 0;
  for (int e = 0; e < P.m; e++) {
    int u = P.eu[e], v = P.ev[e];
    if (u < 0 || v < 0 || u >= P.n || v >= P.n || u == v) return fail(nullptr, BBTN_EINVAL, "edge " + std::to_string(e) + " is malformed");
    seen.push_back({std::min(u, v), std::max(u, v)});
  }
  std::sort(seen.begin(), seen.end());
  for (size_t i = 1; i < seen.size(); i++) if (seen[i] == seen[i - 1]) return fail(nullptr, BBTN_EINVAL, "duplicate edge");
  P.ew.resize(P.m); P.vw.resize(P.n);
  for (int e = 0; e < P.m; e++) { P.ew[e] = (P.kind == BBTN_ISING && d->edge_w) ? d->edge_w[e] : 1; if (P.kind == BBTN_ISING) range += std::abs((int64_t)P.ew[e]); }
  for (int i = 0; i < P.n; i++) {
    P.vw[i] = d->vertex_w ? d->vertex_w[i] : (P.kind == BBTN_ISING ? 0 : 1);
    range += std::abs((int64_t)P.vw[i]);
  }
  if (range > BBTN_ENERGY_LIMIT) return fail(nullptr, BBTN_ERANGE, "sum of |couplings| + |weights| exceeds 2^28");
  P.energy_range = range;
  if (d->tree_l || d->n_steps > 0) {
    if (!d->tree_l || !d->tree_r || d->n_steps != P.n + P.m - 1)
      return fail(nullptr, BBTN_EINVAL, "tree must have n_edges + n_vertices - 1 steps");
    P.tree_l.assign(d->tree_l, d->tree_l + d->n_steps); P.tree_r.assign(d->tree_r, d->tree_r + d->n_steps);
  }
  P.max_elements = d->max_elements_per_leaf > 0 ? d->max_elements_per_leaf : ((int64_t)1 << 28);
  h->force_mode = (d->flags & BBTN_FORCE_STREAMING) ? 1 : ((d->flags & BBTN_FORCE_TILED) ? 2 : 0);
  if (d->flags & BBTN_SEARCH_ONLY) {
    if (d->flags & BBTN_COUNT_CRT) return fail(nullptr, BBTN_EINVAL, "BBTN_SEARCH_ONLY excludes BBTN_COUNT_CRT");
  }
  // validate the tree once on the unsliced network
  if (!P.tree_l.empty()) {
    Plan tmp; std::string err;
    int rc = make_plan(P, {}, h->force_mode, false, tmp, err);
    if (rc) return fail(nullptr, rc, err);
  }
  *out = h.release();
  return BBTN_OK;
}

void bbtn_destroy(bbtn_handle *h) { delete h; }

int bbtn_plan_query(bbtn_handle *h, const int32_t *fixed, int32_t n_fixed, int64_t B, bbtn_plan_info *info) {
  if (!h || !info || B < 1) return fail(h, BBTN_EINVAL, "null argument");
  DevPlan *dp = nullptr;
  int rc = get_plan(h, fixed, n_fixed, false, &dp);
  if (rc) return rc;
  const Plan &pl = dp->plan;
  std::memset(info, 0, sizeof(*info));
  info->n_nodes = pl.n_nodes; info->n_variant_nodes = pl.n_variant_nodes; info->max_rank = pl.max_rank;
  for (const Step &s : pl.steps) {
    if (s.kind == STEP_GEMM) info->n_gemm_tiled++;
    else if (s.kind == STEP_ABSORB) info->n_absorb++;
    else if (s.kind == STEP_PERMUTE) info->n_permute++;
    else info->n_trace++;
  }
  info->rho = pl.rho;
  info->fma_variant = pl.fma_variant; info->fma_invariant = pl.fma_invariant;
  const bool search = (h->P.flags & BBTN_SEARCH_ONLY) != 0;      // 4 B per element instead of 12
  info->bytes_per_call = (pl.bytes_variant * (double)B + pl.bytes_invariant) / (search ? 3.0 : 1.0);
  info->workspace_bytes = (pl.arena_variant_elems * B + pl.arena_invariant_elems) * (search ? 4 : 12);
  int n_var = 0, n_inv = 0;
  for (const InputRec &r : pl.inputs) if (r.rank > 0) (r.variant ? n_var : n_inv)++;
  // K1: variant tensors, invariant tensors, offset[b]; K4: finalize
  info->n_kernel_launches = (int32_t)pl.steps.size() + (n_var > 0) + (n_inv > 0) + 2;
  if (dp->hybrid == 1 && B <= dp->hyb_max_B)             // small subtrees run as one or two shared-memory prologue launches
    info->n_kernel_launches = (int32_t)dp->hyb_big.size() + !dp->hyb[0].steps.empty() + !dp->hyb[1].steps.empty() + (n_var > 0) + (n_inv > 0) + 2;
  return BBTN_OK;
}

int bbtn_contract_batch(bbtn_handle *h, const int32_t *fixed, int32_t n_fixed, const uint8_t *assign, int64_t B,
                        int32_t *energy, uint64_t *count, uint32_t *count_mod, void *stream) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  if (B < 1 || !energy || (!count && !(h->P.flags & BBTN_SEARCH_ONLY)) || (n_fixed > 0 && !assign))
    return fail(h, BBTN_EINVAL, "bad batch arguments");
  const bool crt = (h->P.flags & BBTN_COUNT_CRT) != 0;
  if (count_mod && !crt) return fail(h, BBTN_EINVAL, "count_mod needs a handle built with BBTN_COUNT_CRT");
  if (!have_device()) return fail(h, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  DevPlan *dp = nullptr;
  int rc = get_plan(h, fixed, n_fixed, true, &dp);
  if (rc) return rc;
  return bbtn::run_plan(h, dp, assign, B, energy, count, count_mod, true, stream);
}

}  // extern "C"

// Run one planned contraction (K1 -> K2/K3 -> K4) for B leaves; shared by bbtn_contract_batch (cached
// plans, CUDA-graph replay) and the branching driver (one-leaf plans on the handle's scratch buffers).
int bbtn::run_plan(bbtn_handle *h, DevPlan *dp, const uint8_t *assign, int64_t B, int32_t *energy, uint64_t *count,
                   uint32_t *count_mod, bool allow_graph, void *stream) {
  const bool crt = (h->P.flags & BBTN_COUNT_CRT) != 0;
  const int32_t n_fixed = (int32_t)dp->plan.fixed.size();
  int rc;
  if ((rc = upload_tables(h, dp))) return rc;
  const bool dev_io = (h->P.flags & BBTN_IO_DEVICE) != 0;
  // With host pointers the library owns the device-side batch buffers, so the launched batch is rounded up to
  // a power of two (padding leaves = assignment 0, results dropped): the CUDA graph of this fixed set is then
  // captured once per size class instead of once per distinct B (the host B&B loop sends ragged batches).
  const int64_t B_user = B;
  if ((rc = prepare_fused(h, dp))) return rc;
  if (!dev_io && dp->fused != 1) {
    int64_t bp = 1; while (bp < B) bp <<= 1;
    // pad only when the padded arena fits; a ragged B just above a power of two must not turn into ENOMEM
    size_t free_b = 0, total_b = 0;
    if (bp <= dp->B_cap || (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess &&
                            (double)dp->plan.arena_variant_elems * (double)bp * 12.0 <= (double)free_b + (double)dp->var_e.bytes + (double)dp->var_c.bytes))
      B = bp;
  }
  if ((rc = ensure_batch(h, dp, B, !dev_io))) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const uint8_t *d_assign = assign; int32_t *d_energy = energy; uint64_t *d_count = count; uint32_t *d_mod = count_mod;
  if (!dev_io) {
    d_assign = (const uint8_t *)dp->assign.p; d_energy = (int32_t *)dp->energy.p; d_count = (uint64_t *)dp->count.p;
    d_mod = count_mod ? (uint32_t *)dp->count_mod.p : nullptr;
    if (n_fixed > 0) {
      CUDA_TRY(h, cudaMemcpyAsync(dp->assign.p, assign, (size_t)B_user * n_fixed, cudaMemcpyHostToDevice, st));
      if (B > B_user)
        CUDA_TRY(h, cudaMemsetAsync((char *)dp->assign.p + (size_t)B_user * n_fixed, 0, (size_t)(B - B_user) * n_fixed, st));
    }
  }
  const bool search = (h->P.flags & BBTN_SEARCH_ONLY) != 0;
  // CRT mode: a second pass with both prime residues in one 64-bit count (every kernel of the path has that form; K2
  // moves the pair as a 64-bit word)
  const int rings[2] = {search ? (int)RING_NONE : (int)RING_U64, (int)RING_P12};
  const int n_rings = (!search && crt && d_mod) ? 2 : 1;
  const bool use_graph = allow_graph && !(h->P.flags & BBTN_NO_GRAPH) && dp->plan.steps.size() >= 8;
  for (int ring = 0; ring < n_rings; ring++) {             // shared-memory opt-in of the kernels that keep a leaf's tensors on chip
    if (dp->fused == 1) configure_fused_tree(rings[ring], dp->plan.max_rank);
    if (dp->hybrid == 1) for (auto &g : dp->hyb) if (!g.steps.empty()) configure_fused_tree(rings[ring], g.max_rank);
  }
  if (dp->fused == 1) {
    const Plan &pl = dp->plan;
    for (int ring = 0; ring < n_rings; ring++)
      launch_fused_tree(h->P.kind, (const InputRec *)dp->inputs.p, (const int32_t *)dp->list_build.p, dp->n_build,
                        (const int32_t *)dp->list_scalar.p, dp->n_scalar, d_assign, n_fixed, B, (const FusedStep *)dp->fused_steps.p,
                        (int)pl.steps.size(), dp->fused_arena, (int)pl.arena_variant_elems, (int)pl.result_offset,
                        d_energy, d_count, d_mod, rings[ring], pl.max_rank, st);
  } else if (!use_graph) {
    for (int ring = 0; ring < n_rings; ring++) enqueue_ring(h, dp, B, d_assign, d_energy, d_count, d_mod, rings[ring], st);
  } else {
    const void *io[4] = {d_assign, d_energy, d_count, d_mod};
    const bool stale = dp->graph_B != B || (int)dp->graphs.size() != n_rings || std::memcmp(io, dp->graph_io, sizeof(io)) != 0;
    if (stale) {
      for (auto g : dp->graphs) if (g) cudaGraphExecDestroy(g);
      dp->graphs.clear();
      cudaStream_t cs;
      CUDA_TRY(h, cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
      cudaError_t ce = cudaSuccess;
      for (int ring = 0; ring < n_rings && ce == cudaSuccess; ring++) {
        cudaGraph_t g = nullptr; cudaGraphExec_t ge = nullptr;
        if ((ce = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal)) != cudaSuccess) break;
        enqueue_ring(h, dp, B, d_assign, d_energy, d_count, d_mod, rings[ring], cs);
        ce = cudaStreamEndCapture(cs, &g);          // always ends the capture, also after a failed launch
        if (ce == cudaSuccess) ce = cudaGraphInstantiate(&ge, g, 0);
        if (g) cudaGraphDestroy(g);
        if (ce == cudaSuccess) dp->graphs.push_back(ge);
      }
      cudaStreamDestroy(cs);
      if (ce != cudaSuccess) {
        for (auto g : dp->graphs) if (g) cudaGraphExecDestroy(g);
        dp->graphs.clear(); dp->graph_B = -1;
        CUDA_TRY(h, ce);
      }
      dp->graph_B = B; std::memcpy(dp->graph_io, io, sizeof(io));
    }
    for (auto ge : dp->graphs) CUDA_TRY(h, cudaGraphLaunch(ge, st));
  }
  CUDA_TRY(h, cudaGetLastError());
  if (!dev_io) {
    // stage into temporaries so that outputs stay untouched on error
    std::vector<int32_t> te((size_t)B_user); std::vector<uint64_t> tc((size_t)B_user); std::vector<uint32_t> tm(count_mod ? (size_t)B_user * 2 : 0);
    CUDA_TRY(h, cudaMemcpyAsync(te.data(), d_energy, (size_t)B_user * 4, cudaMemcpyDeviceToHost, st));
    if (count) CUDA_TRY(h, cudaMemcpyAsync(tc.data(), d_count, (size_t)B_user * 8, cudaMemcpyDeviceToHost, st));
    if (count_mod) CUDA_TRY(h, cudaMemcpyAsync(tm.data(), d_mod, (size_t)B_user * 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(h, cudaStreamSynchronize(st));
    std::memcpy(energy, te.data(), (size_t)B_user * 4);
    if (count) std::memcpy(count, tc.data(), (size_t)B_user * 8);
    if (count_mod) std::memcpy(count_mod, tm.data(), (size_t)B_user * 8);
  }
  return BBTN_OK;
}

extern "C" {

int bbtn_tropical_gemm_batched(int64_t batch, int32_t M, int32_t N, int32_t K, const int32_t *Ae, const uint64_t *Ac,
                               const int32_t *Be, const uint64_t *Bc, int32_t *Ce, uint64_t *Cc,
                               int64_t strideA, int64_t strideB, int64_t strideC, int32_t count_bits, int32_t energy_bits,
                               void *stream) {
  if (batch < 1 || M < 1 || N < 1 || K < 1 || !Ae || !Ac || !Be || !Bc || !Ce || !Cc || strideA < 0 || strideB < 0 || strideC < 0)
    return fail(nullptr, BBTN_EINVAL, "bad GEMM arguments");
  if (batch > 1 && strideC < (int64_t)M * N) return fail(nullptr, BBTN_EINVAL, "strideC overlaps outputs");
  int rc = check_gemm_shape(batch, M, N, count_bits, energy_bits);
  if (rc) return rc;
  if (!have_device()) return fail(nullptr, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  if (g_debug_checks && (rc = check_gemm_operands(batch, M, N, K, Ae, Ac, Be, Bc, strideA, strideB, count_bits, energy_bits, (cudaStream_t)stream))) return rc;
  launch_gemm_tiled(batch, 1, M, N, K, 0, Ae, Ac, Be, Bc, Ce, Cc, strideA, strideB, strideC, RING_U64, count_bits, energy_bits,
                    (cudaStream_t)stream);
  CUDA_TRY(nullptr, cudaGetLastError());
  return BBTN_OK;
}

int bbtn_maxplus_gemm_batched(int64_t batch, int32_t M, int32_t N, int32_t K, const int32_t *A, const int32_t *B, int32_t *C,
                              int64_t strideA, int64_t strideB, int64_t strideC, int32_t energy_bits, void *stream) {
  if (batch < 1 || M < 1 || N < 1 || K < 1 || !A || !B || !C || strideA < 0 || strideB < 0 || strideC < 0)
    return fail(nullptr, BBTN_EINVAL, "bad GEMM arguments");
  if (batch > 1 && strideC < (int64_t)M * N) return fail(nullptr, BBTN_EINVAL, "strideC overlaps outputs");
  int rc = check_gemm_shape(batch, M, N, 1, energy_bits);
  if (rc) return rc;
  if (!have_device()) return fail(nullptr, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  if (g_debug_checks && (rc = check_gemm_operands(batch, M, N, K, A, nullptr, B, nullptr, strideA, strideB, 64, energy_bits, (cudaStream_t)stream))) return rc;
  launch_gemm_maxplus(batch, 1, M, N, K, 0, A, B, C, strideA, strideB, strideC, energy_bits, (cudaStream_t)stream);
  CUDA_TRY(nullptr, cudaGetLastError());
  return BBTN_OK;
}

int bbtn_tropical_gemm_batched_host(int64_t batch, int32_t M, int32_t N, int32_t K, const int32_t *Ae, const uint64_t *Ac,
                                    const int32_t *Be, const uint64_t *Bc, int32_t *Ce, uint64_t *Cc,
                                    int64_t strideA, int64_t strideB, int64_t strideC, int32_t count_bits, int32_t energy_bits,
                                    void *stream) {
  if (batch < 1 || M < 1 || N < 1 || K < 1 || !Ae || !Ac || !Be || !Bc || !Ce || !Cc || strideA < 0 || strideB < 0 || strideC < 0)
    return fail(nullptr, BBTN_EINVAL, "bad GEMM arguments");
  if (batch > 1 && strideC < (int64_t)M * N) return fail(nullptr, BBTN_EINVAL, "strideC overlaps outputs");
  if ((strideA && strideA < (int64_t)M * K) || (strideB && strideB < (int64_t)K * N))
    return fail(nullptr, BBTN_EINVAL, "operand stride smaller than the operand");
  { int rc = check_gemm_shape(batch, M, N, count_bits, energy_bits); if (rc) return rc; }
  if (!have_device()) return fail(nullptr, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  static thread_local DevBuf st_e[3], st_c[3];
  cudaStream_t st = (cudaStream_t)stream;
  const size_t nA = (size_t)(strideA ? (batch - 1) * strideA : 0) + (size_t)M * K;
  const size_t nB = (size_t)(strideB ? (batch - 1) * strideB : 0) + (size_t)K * N;
  const size_t nC = (size_t)(batch - 1) * strideC + (size_t)M * N;
  const size_t n[3] = {nA, nB, nC};
  for (int i = 0; i < 3; i++) { CUDA_TRY(nullptr, st_e[i].ensure(n[i] * 4)); CUDA_TRY(nullptr, st_c[i].ensure(n[i] * 8)); }
  // The batch is cut into chunks that flow through three internal streams -- host->device copies, K3, device->host
  // copies -- so the PCIe transfers of chunk c+1 / c-1 overlap the GEMM of chunk c (pinned host memory needed for
  // the overlap; pageable memory still works, serialised by the driver).  Shared operands (stride 0) go up once.
  static thread_local cudaStream_t s_in = nullptr, s_k = nullptr, s_out = nullptr;
  static thread_local cudaEvent_t ev_start = nullptr, ev_in[16], ev_k[16], ev_done = nullptr;
  if (!s_in) {
    CUDA_TRY(nullptr, cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
    CUDA_TRY(nullptr, cudaStreamCreateWithFlags(&s_k, cudaStreamNonBlocking));
    CUDA_TRY(nullptr, cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
    CUDA_TRY(nullptr, cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
    CUDA_TRY(nullptr, cudaEventCreateWithFlags(&ev_done, cudaEventDisableTiming));
    for (int i = 0; i < 16; i++) {
      CUDA_TRY(nullptr, cudaEventCreateWithFlags(&ev_in[i], cudaEventDisableTiming));
      CUDA_TRY(nullptr, cudaEventCreateWithFlags(&ev_k[i], cudaEventDisableTiming));
    }
  }
  const int n_chunks = (int)std::min<int64_t>(16, std::max<int64_t>(1, batch / 4));   // >= 4 entries per chunk; short chunks keep the tail (last GEMM + copy-out) small
  int32_t *dAe = (int32_t *)st_e[0].p, *dBe = (int32_t *)st_e[1].p, *dCe = (int32_t *)st_e[2].p;
  uint64_t *dAc = (uint64_t *)st_c[0].p, *dBc = (uint64_t *)st_c[1].p, *dCc = (uint64_t *)st_c[2].p;
  CUDA_TRY(nullptr, cudaEventRecord(ev_start, st));
  CUDA_TRY(nullptr, cudaStreamWaitEvent(s_in, ev_start, 0));
  CUDA_TRY(nullptr, cudaStreamWaitEvent(s_out, ev_start, 0));   // earlier work on st may still read the staging buffers
  if (!strideA) {
    CUDA_TRY(nullptr, cudaMemcpyAsync(dAe, Ae, (size_t)M * K * 4, cudaMemcpyHostToDevice, s_in));
    CUDA_TRY(nullptr, cudaMemcpyAsync(dAc, Ac, (size_t)M * K * 8, cudaMemcpyHostToDevice, s_in));
  }
  if (!strideB) {
    CUDA_TRY(nullptr, cudaMemcpyAsync(dBe, Be, (size_t)K * N * 4, cudaMemcpyHostToDevice, s_in));
    CUDA_TRY(nullptr, cudaMemcpyAsync(dBc, Bc, (size_t)K * N * 8, cudaMemcpyHostToDevice, s_in));
  }
  for (int c = 0; c < n_chunks; c++) {
    const int64_t b0 = batch * c / n_chunks, b1 = batch * (c + 1) / n_chunks, nb = b1 - b0;
    if (strideA) {
      const size_t off = (size_t)b0 * strideA, len = (size_t)(nb - 1) * strideA + (size_t)M * K;
      CUDA_TRY(nullptr, cudaMemcpyAsync(dAe + off, Ae + off, len * 4, cudaMemcpyHostToDevice, s_in));
      CUDA_TRY(nullptr, cudaMemcpyAsync(dAc + off, Ac + off, len * 8, cudaMemcpyHostToDevice, s_in));
    }
    if (strideB) {
      const size_t off = (size_t)b0 * strideB, len = (size_t)(nb - 1) * strideB + (size_t)K * N;
      CUDA_TRY(nullptr, cudaMemcpyAsync(dBe + off, Be + off, len * 4, cudaMemcpyHostToDevice, s_in));
      CUDA_TRY(nullptr, cudaMemcpyAsync(dBc + off, Bc + off, len * 8, cudaMemcpyHostToDevice, s_in));
    }
    CUDA_TRY(nullptr, cudaEventRecord(ev_in[c], s_in));
    CUDA_TRY(nullptr, cudaStreamWaitEvent(s_k, ev_in[c], 0));
    if (g_debug_checks) {
      int rc = check_gemm_operands(nb, M, N, K, dAe + b0 * strideA, dAc + b0 * strideA, dBe + b0 * strideB, dBc + b0 * strideB,
                                   strideA, strideB, count_bits, energy_bits, s_k);
      if (rc) { cudaStreamSynchronize(s_in); cudaStreamSynchronize(s_out); return rc; }
    }
    launch_gemm_tiled(nb, 1, M, N, K, 0, dAe + b0 * strideA, dAc + b0 * strideA, dBe + b0 * strideB, dBc + b0 * strideB,
                      dCe + b0 * strideC, dCc + b0 * strideC, strideA, strideB, strideC, RING_U64, count_bits, energy_bits, s_k);
    CUDA_TRY(nullptr, cudaGetLastError());
    CUDA_TRY(nullptr, cudaEventRecord(ev_k[c], s_k));
    CUDA_TRY(nullptr, cudaStreamWaitEvent(s_out, ev_k[c], 0));
    const size_t off = (size_t)b0 * strideC, len = (size_t)(nb - 1) * strideC + (size_t)M * N;
    CUDA_TRY(nullptr, cudaMemcpyAsync(Ce + off, dCe + off, len * 4, cudaMemcpyDeviceToHost, s_out));
    CUDA_TRY(nullptr, cudaMemcpyAsync(Cc + off, dCc + off, len * 8, cudaMemcpyDeviceToHost, s_out));
  }
  CUDA_TRY(nullptr, cudaEventRecord(ev_done, s_out));
  CUDA_TRY(nullptr, cudaStreamWaitEvent(st, ev_done, 0));
  CUDA_TRY(nullptr, cudaStreamSynchronize(st));
  return BBTN_OK;
}

int bbtn_permute_batched(int32_t rank, const int32_t *perm, int64_t batch, const int32_t *src_e, const uint64_t *src_c,
                         int32_t *dst_e, uint64_t *dst_c, void *stream) {
  if (rank < 0 || rank > 30 || batch < 1 || (rank > 0 && !perm) || !src_e || !src_c || !dst_e || !dst_c)
    return fail(nullptr, BBTN_EINVAL, "bad permute arguments");
  uint32_t seen = 0;
  for (int j = 0; j < rank; j++) {
    if (perm[j] < 0 || perm[j] >= rank || (seen >> perm[j]) & 1u) return fail(nullptr, BBTN_EINVAL, "perm is not a permutation");
    seen |= 1u << perm[j];
  }
  if (!have_device()) return fail(nullptr, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  launch_permute(rank, perm, batch, src_e, src_c, dst_e, dst_c, RING_U64, (cudaStream_t)stream);
  CUDA_TRY(nullptr, cudaGetLastError());
  return BBTN_OK;
}

int bbtn_set_debug_checks(int32_t on) {
  const int prev = g_debug_checks ? 1 : 0;
  g_debug_checks = on != 0;
  return prev;
}

// CRT over the pairwise coprime moduli 2^64, P1, P2 (Garner's form): x = c64 + 2^64 * (t1 + P1 * t2).
int bbtn_crt_combine(uint64_t c64, uint32_t r1, uint32_t r2, uint64_t out[2]) {
  if (!out || r1 >= BBTN_P1 || r2 >= BBTN_P2) return fail(nullptr, BBTN_EINVAL, "bad crt_combine arguments");
  auto powmod = [](uint64_t b, uint64_t e, uint64_t p) { uint64_t r = 1; b %= p; for (; e; e >>= 1, b = b * b % p) if (e & 1) r = r * b % p; return r; };
  const uint64_t p1 = BBTN_P1, p2 = BBTN_P2;
  const uint64_t two64_p1 = (((uint64_t)1 << 32) % p1) * (((uint64_t)1 << 32) % p1) % p1;
  const uint64_t two64_p2 = (((uint64_t)1 << 32) % p2) * (((uint64_t)1 << 32) % p2) % p2;
  // t1 = (r1 - c64) / 2^64 mod P1     (inverse by Fermat: P1 is prime)
  const uint64_t t1 = (r1 + p1 - c64 % p1) % p1 * powmod(two64_p1, p1 - 2, p1) % p1;
  // x1 = c64 + 2^64 t1;  t2 = (r2 - x1) / (2^64 P1) mod P2
  const uint64_t x1_p2 = (c64 % p2 + two64_p2 * (t1 % p2)) % p2;
  const uint64_t m_p2 = two64_p2 * (p1 % p2) % p2;
  const uint64_t t2 = (r2 + p2 - x1_p2) % p2 * powmod(m_p2, p2 - 2, p2) % p2;
  out[0] = c64;
  out[1] = t1 + p1 * t2;            // < P1 * P2 < 2^62
  return BBTN_OK;
}

int bbtn_int32_microbench(int32_t which, int32_t iters, double *ms, double *ops, void *stream) {
  if (which < 0 || which > 15 || iters < 1 || !ms || !ops) return fail(nullptr, BBTN_EINVAL, "bad microbench arguments");
  if (!have_device()) return fail(nullptr, BBTN_ECUDA, "no CUDA device");
  int rc = run_microbench(which, iters, ms, ops, (cudaStream_t)stream);
  if (rc) return fail(nullptr, BBTN_ECUDA, "microbenchmark failed");
  return BBTN_OK;
}

}  // extern "C"
