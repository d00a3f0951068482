// branching.cu -- host side of BBTN proper: non-uniform branching driven by the
// memory-overflow measure rho of Eq. 4, leaves contracted on the device one plan at a time.
//
//   rho(T) = sum over the tensors of the contraction tree of max(0, log2|T| - log2 T_target)    (Eq. 4)
//
// Branching rule generator (the paper's optimal-branching rule search and inference rules are in its
// missing supplement / ref [46]; DESIGN.md "readings" A23): one vertex v per branching,
//   MIS   D = { (v = 0),  (v = 1 and every free neighbour of v = 0) }      complete: a set either holds v or not;
//                                                                          orthogonal: the two differ in s_v
//   Ising D = { (s_v = 0), (s_v = 1) }
// and v is the free vertex that minimises the branching factor gamma, the root of
//   gamma^rho(T) = sum_i gamma^rho(T_i)
// i.e. of 1 = gamma^-d0 + gamma^-d1 with d_i = rho(T) - rho(T_i).  A branch with rho = 0 whose plan fits the
// device-memory budget is a leaf: it is planned on the unsliced tree with its fixed indices deleted and
// contracted by K1..K4 (run_plan), and the leaf results are (+)-accumulated ("summing the
// contractions of each branch").  Plain C++; every arithmetic step on tensors runs in the kernels.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "handle.h"

using namespace bbtn;

namespace {

struct Leaf { std::vector<int32_t> fixed; std::vector<uint8_t> val; };

struct Brancher {
  bbtn_handle *h;
  const Problem *P;                               // problem with the tree filled in
  int t;                                          // log2 T_target
  int64_t mem_budget;                             // bytes a leaf's arena may take (0 = unlimited)
  int64_t max_leaves;
  std::vector<std::vector<int32_t>> node_labels;  // output labels of every launched tree node (unsliced)
  std::vector<std::vector<int32_t>> nodes_of;     // vertex -> nodes carrying it
  std::vector<std::vector<int32_t>> adj;
  std::vector<int> rank;                          // current rank of every node (fixed labels deleted)
  std::vector<int8_t> val;                        // -1 free, else the fixed value
  std::vector<int32_t> trail;                     // fixed vertices in the order they were fixed
  std::vector<int> cnt;                           // scratch, per node
  int64_t n_branch_nodes = 0, max_fixed = 0, rho_root = 0;
  std::vector<Leaf> *sink = nullptr;              // collect leaves (host-only enumeration) ...
  // ... or contract them as they appear
  bool contract = false; void *stream = nullptr; bool want_mod = false;
  bool have_best = false; int32_t best = BBTN_NEG_INF; uint64_t c64 = 0, m1 = 0, m2 = 0;
  int64_t n_leaves = 0;
  double leaf_bytes = 0, leaf_fma = 0;

  int init(std::string &err) {
    Plan pl;
    int rc = make_plan(*P, {}, h->force_mode, false, pl, err, true, true);
    if (rc) return rc;
    node_labels.swap(pl.node_labels);
    nodes_of.assign(P->n, {});
    rank.resize(node_labels.size());
    for (size_t k = 0; k < node_labels.size(); k++) {
      rank[k] = (int)node_labels[k].size();
      for (int v : node_labels[k]) nodes_of[v].push_back((int32_t)k);
    }
    adj.assign(P->n, {});
    for (int e = 0; e < P->m; e++) { adj[P->eu[e]].push_back(P->ev[e]); adj[P->ev[e]].push_back(P->eu[e]); }
    val.assign(P->n, -1);
    cnt.assign(node_labels.size(), 0);
    return 0;
  }
  int64_t rho(int tt) const {
    int64_t r = 0;
    for (int k : rank) r += std::max(0, k - tt);
    return r;
  }
  void fix(int v, int x) { val[v] = (int8_t)x; trail.push_back(v); for (int k : nodes_of[v]) rank[k]--; }
  void unfix_to(size_t mark) {
    while (trail.size() > mark) { int v = trail.back(); trail.pop_back(); val[v] = -1; for (int k : nodes_of[v]) rank[k]++; }
  }
  // decrease of rho (threshold tt) when the free vertices in S are fixed
  int64_t gain(const std::vector<int32_t> &S, int tt) {
    int64_t g = 0;
    for (int u : S) for (int k : nodes_of[u]) if (rank[k] > tt) cnt[k]++;
    for (int u : S) for (int k : nodes_of[u]) if (cnt[k]) { g += std::min(cnt[k], rank[k] - tt); cnt[k] = 0; }
    return g;
  }
  void branch_set(int v, std::vector<int32_t> &S1) const {
    S1.clear(); S1.push_back(v);
    if (P->kind == BBTN_MIS) for (int u : adj[v]) if (val[u] < 0) S1.push_back(u);
  }
  static double gamma_of(int64_t d0, int64_t d1) {
    if (d0 <= 0 || d1 <= 0) return 1e30;
    double lo = 1.0, hi = 2.0;                    // f(x) = x^-d0 + x^-d1 - 1 decreases; f(1) = 1, f(2) <= 0
    for (int it = 0; it < 60; it++) {
      double x = 0.5 * (lo + hi);
      (std::pow(x, -(double)d0) + std::pow(x, -(double)d1) > 1.0 ? lo : hi) = x;
    }
    return hi;
  }
  // the free vertex with the smallest branching factor at threshold tt; -1 if no vertex lowers rho
  int pick(int tt) {
    std::vector<char> cand(P->n, 0);
    for (size_t k = 0; k < node_labels.size(); k++)
      if (rank[k] > tt) for (int v : node_labels[k]) if (val[v] < 0) cand[v] = 1;
    int bestv = -1; double bg = 1e31; int64_t bsum = -1;
    std::vector<int32_t> S0(1), S1;
    for (int v = 0; v < P->n; v++) {
      if (!cand[v]) continue;
      S0[0] = v;
      const int64_t d0 = gain(S0, tt);
      branch_set(v, S1);
      const int64_t d1 = S1.size() == 1 ? d0 : gain(S1, tt);
      const double g = gamma_of(d0, d1);
      if (g < bg - 1e-12 || (std::fabs(g - bg) <= 1e-12 && d0 + d1 > bsum)) { bestv = v; bg = g; bsum = d0 + d1; }
    }
    return bestv;
  }

  int emit_leaf(const Plan *pl) {
    n_leaves++;
    max_fixed = std::max<int64_t>(max_fixed, (int64_t)trail.size());
    if (pl) { leaf_bytes += pl->bytes_variant + pl->bytes_invariant; leaf_fma += pl->fma_variant + pl->fma_invariant; }
    if (max_leaves > 0 && n_leaves > max_leaves)
      return fail(h, BBTN_ESHAPE, "branching needs more than max_leaves = " + std::to_string(max_leaves) + " leaves");
    if (sink) {
      Leaf lf; lf.fixed = trail;
      for (int v : trail) lf.val.push_back((uint8_t)val[v]);
      sink->push_back(std::move(lf));
    }
    if (!contract) return BBTN_OK;
    std::vector<uint8_t> a;
    for (int v : trail) a.push_back((uint8_t)val[v]);
    int32_t e; uint64_t c; uint32_t cm[2] = {0, 0};
    DevPlan *dp = h->scratch.get();
    int rc = run_plan(h, dp, a.data(), 1, &e, &c, want_mod ? cm : nullptr, false, stream);
    if (rc) return rc;
    if (e == BBTN_NEG_INF) return BBTN_OK;
    const bool better = !have_best || (P->kind == BBTN_ISING ? e < best : e > best);
    if (better) { best = e; c64 = 0; m1 = m2 = 0; have_best = true; }
    if (e == best) { c64 += c; m1 = (m1 + cm[0]) % BBTN_P1; m2 = (m2 + cm[1]) % BBTN_P2; }
    return BBTN_OK;
  }

  int recurse(int tt) {
    int v = -1;
    if (rho(tt) > 0) v = pick(tt);
    else {
      // rho = 0: plan the leaf on the unsliced tree; if its arena exceeds the budget, keep branching
      // against a tighter threshold
      DevPlan *dp = h->scratch.get();
      std::string err;
      int rc = make_plan(*P, trail, h->force_mode, false, dp->plan, err, true, false);
      if (rc) return fail(h, rc, err);
      dp->tables_ready = false; dp->B_cap = 0; dp->graph_B = -1; dp->fused = -1;
      const int64_t bytes = dp->plan.arena_variant_elems * 12;
      if (mem_budget <= 0 || bytes <= mem_budget || tt <= 4) return emit_leaf(&dp->plan);
      while (tt > 4 && rho(tt) == 0) tt--;
      if (rho(tt) == 0) return emit_leaf(&dp->plan);
      v = pick(tt);
    }
    if (v < 0) return fail(h, BBTN_ESHAPE, "no branching vertex lowers rho (internal)");
    n_branch_nodes++;
    const size_t mark = trail.size();
    std::vector<int32_t> S1;
    branch_set(v, S1);
    // branch 1: v = 1 (MIS: its free neighbours = 0)
    fix(v, 1);
    for (size_t i = 1; i < S1.size(); i++) fix(S1[i], 0);
    int rc = recurse(tt);
    unfix_to(mark);
    if (rc) return rc;
    // branch 0: v = 0
    fix(v, 0);
    rc = recurse(tt);
    unfix_to(mark);
    return rc;
  }
};

int prepare(bbtn_handle *h, int32_t log2_target, int64_t mem_budget, int64_t max_leaves, Brancher &br) {
  if (log2_target < 1 || log2_target > 32) return fail(h, BBTN_EINVAL, "log2_target must be in 1..32");
  if (!h->Pbr) {
    auto P = std::make_unique<Problem>(h->P);
    if (P->tree_l.empty() && P->n + P->m > 1) derive_tree(*P, {}, P->tree_l, P->tree_r);
    h->Pbr = std::move(P);
  }
  if (!h->scratch) h->scratch = std::make_unique<DevPlan>();
  br.h = h; br.P = h->Pbr.get(); br.t = log2_target; br.mem_budget = mem_budget; br.max_leaves = max_leaves;
  std::string err;
  int rc = br.init(err);
  if (rc) return fail(h, rc, err);
  br.rho_root = br.rho(log2_target);
  return BBTN_OK;
}

void write_stats(const Brancher &br, int64_t *stats, double *work) {
  if (stats) { stats[0] = br.n_branch_nodes; stats[1] = br.n_leaves; stats[2] = br.max_fixed; stats[3] = br.rho_root; }
  if (work) { work[0] = br.leaf_fma; work[1] = br.leaf_bytes; }
}

}  // namespace

extern "C" {

int bbtn_branching_leaves(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes, int64_t max_leaves,
                          int64_t cap_leaves, int64_t cap_entries, int64_t *leaf_offsets, int32_t *leaf_vertices,
                          uint8_t *leaf_values, int64_t *stats, double *work) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  Brancher br;
  int rc = prepare(h, log2_target, mem_budget_bytes, max_leaves, br);
  if (rc) return rc;
  std::vector<Leaf> leaves;
  const bool store = leaf_offsets && leaf_vertices && leaf_values;
  if (store) br.sink = &leaves;
  if ((rc = br.recurse(log2_target))) return rc;
  write_stats(br, stats, work);
  if (store) {
    int64_t n_entries = 0;
    for (auto &l : leaves) n_entries += (int64_t)l.fixed.size();
    if ((int64_t)leaves.size() > cap_leaves || n_entries > cap_entries)
      return fail(h, BBTN_EINVAL, "leaf buffers too small: need " + std::to_string(leaves.size()) + " leaves, " +
                                      std::to_string(n_entries) + " entries");
    int64_t o = 0;
    for (size_t i = 0; i < leaves.size(); i++) {
      leaf_offsets[i] = o;
      for (size_t j = 0; j < leaves[i].fixed.size(); j++) { leaf_vertices[o] = leaves[i].fixed[j]; leaf_values[o] = leaves[i].val[j]; o++; }
    }
    leaf_offsets[leaves.size()] = o;
  }
  return BBTN_OK;
}

int bbtn_solve_branching(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes, int64_t max_leaves,
                         int32_t *energy, uint64_t *count, uint32_t *count_mod, int64_t *stats, double *work,
                         void *stream) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  if (!energy || !count) return fail(h, BBTN_EINVAL, "bad solve_branching arguments");
  if (h->P.flags & BBTN_IO_DEVICE) return fail(h, BBTN_EINVAL, "bbtn_solve_branching needs a host-pointer handle");
  const bool crt = (h->P.flags & BBTN_COUNT_CRT) != 0;
  if (count_mod && !crt) return fail(h, BBTN_EINVAL, "count_mod needs a handle built with BBTN_COUNT_CRT");
  if (!have_device()) return fail(h, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  if (mem_budget_bytes <= 0) {
    size_t free_b = 0, total_b = 0;
    CUDA_TRY(h, cudaMemGetInfo(&free_b, &total_b));
    mem_budget_bytes = (int64_t)((double)free_b * 0.94);
  }
  Brancher br;
  int rc = prepare(h, log2_target, mem_budget_bytes, max_leaves, br);
  if (rc) return rc;
  br.contract = true; br.stream = stream; br.want_mod = crt && count_mod != nullptr;
  rc = br.recurse(log2_target);
  // the scratch buffers can be most of the device: give them back
  h->scratch.reset();
  if (rc) return rc;
  *energy = br.have_best ? br.best : BBTN_NEG_INF;
  *count = br.have_best ? br.c64 : 0;
  if (count_mod) { count_mod[0] = (uint32_t)br.m1; count_mod[1] = (uint32_t)br.m2; }
  write_stats(br, stats, work);
  return BBTN_OK;
}

}  // extern "C"
