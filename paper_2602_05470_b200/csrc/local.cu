// local.cu -- BBTN on sub-networks: bbtn_solve_local / bbtn_local_plan_query (include/bbtn.h).
//
// The contraction tree is walked in SSA order.  Where every tensor fits T_target the steps run once.  A
// segment whose tensors overflow T_target is a sub-TN with open legs; it is decomposed by fixing a LOCAL set F
// of variables that are summed inside it ("decomposes a tensor network into multiple smaller
// sub-TNs by fixing a subset of variables"), one contraction per assignment x of F (Eq. 3), and
// its boundary tensor is the (+) over the branches ("summing the contractions of each branch";
// per boundary state the (energy, count) of the interior: the counting form of the boundary-equivalence
// principle, reading A16).  F is chosen to bring Eq. 4's overflow of the segment to
// zero (plan.cpp make_local_plan).  Branches are pruned before they are contracted: infeasible
// ones (MIS: two adjacent variables of F set) and, when the caller supplies regions and an incumbent, those
// whose K5 region bound is strictly worse than the incumbent (reading A14).
// Host logic only: tensors are built, contracted and (+)-accumulated by the kernels (kernels.h).
#include <algorithm>
#include <cmath>
#include <atomic>
#include <cstring>
#include <thread>

#include "handle.h"

using namespace bbtn;

namespace {

struct LocalRun {
  bbtn_handle *h; const Problem *P; LocalPlan *lp; cudaStream_t st;
  int64_t nb_max = 1;                                                    // branches of one stretch contracted per launch sequence
  DevBuf inputs, lists, assign, inv_e, inv_c, var_e, var_c, off_e, off_c, res_e, res_c, res_m;
  std::vector<int32_t> list_host;
  std::vector<int64_t> var_at, inv_at, sc_at;                            // per segment: position of its lists in `lists`
  int64_t gsc_at = 0; int n_gsc = 0;                                     // scalars of the run-once segments, all together
  int64_t n_contracted = 0, n_infeasible = 0, n_pruned = 0, n_launches = 0, n_sequences = 0;
  double fma_done = 0, bytes_done = 0;
  // pruning inputs
  const int32_t *roff = nullptr, *rv = nullptr; int n_regions = 0; bool have_inc = false; int32_t inc = 0;

  int upload() {
    const Plan &pl = lp->plan;
    const bool search = (h->P.flags & BBTN_SEARCH_ONLY) != 0;
    CUDA_TRY(h, inputs.ensure(pl.inputs.size() * sizeof(InputRec)));
    CUDA_TRY(h, cudaMemcpy(inputs.p, pl.inputs.data(), pl.inputs.size() * sizeof(InputRec), cudaMemcpyHostToDevice));
    for (const LocalSeg &s : lp->segs) {
      var_at.push_back((int64_t)list_host.size()); list_host.insert(list_host.end(), s.list_var.begin(), s.list_var.end());
      inv_at.push_back((int64_t)list_host.size()); list_host.insert(list_host.end(), s.list_inv.begin(), s.list_inv.end());
      sc_at.push_back((int64_t)list_host.size());
      if (!s.fixed.empty()) list_host.insert(list_host.end(), s.list_scalar.begin(), s.list_scalar.end());
    }
    gsc_at = (int64_t)list_host.size();
    for (const LocalSeg &s : lp->segs) if (s.fixed.empty()) { list_host.insert(list_host.end(), s.list_scalar.begin(), s.list_scalar.end()); n_gsc += (int)s.list_scalar.size(); }
    CUDA_TRY(h, lists.upload(list_host));
    CUDA_TRY(h, inv_e.ensure((size_t)pl.arena_invariant_elems * 4));
    CUDA_TRY(h, inv_c.ensure(search ? 0 : (size_t)pl.arena_invariant_elems * 8));
    CUDA_TRY(h, var_e.ensure((size_t)pl.arena_variant_elems * (size_t)nb_max * 4));
    CUDA_TRY(h, var_c.ensure(search ? 0 : (size_t)pl.arena_variant_elems * (size_t)nb_max * 8));
    CUDA_TRY(h, off_e.ensure((size_t)(nb_max + 2) * 4)); CUDA_TRY(h, off_c.ensure((size_t)(nb_max + 2) * 8));
    CUDA_TRY(h, res_e.ensure(4)); CUDA_TRY(h, res_c.ensure(8)); CUDA_TRY(h, res_m.ensure(8));
    return BBTN_OK;
  }

  // the steps of one segment for nb branches at once; xs = their assignment rows [nb][|F|] on the device
  void launch_steps(const LocalSeg &s, int64_t nb, const uint8_t *xs, int ring) {
    const Plan &pl = lp->plan;
    int32_t *ve = (int32_t *)var_e.p, *ie = (int32_t *)inv_e.p;
    char *vc = (char *)var_c.p, *ic = (char *)inv_c.p;
    const size_t csz = ring_count_bytes(ring);
    // a view (x) and an invariant tensor live in the invariant arena; a variant tensor is [nb][2^rank] at off * nb
    auto pe = [&](int v, int x, int64_t off) { return (v && !x) ? ve + off * nb : ie + off; };
    auto pc = [&](int v, int x, int64_t off) { return (void *)((v && !x) ? vc + (size_t)off * nb * csz : ic + (size_t)off * csz); };
    for (int q = s.step_begin; q < s.step_end; q++) {
      const Step &sp = pl.steps[q];
      const int64_t n = sp.variant ? nb : 1;
      const uint8_t *x = (sp.n_slice && (sp.xA || sp.xB)) ? xs : nullptr;
      if (sp.kind == STEP_ABSORB)
        launch_absorb(sp, n, pe(sp.vA, sp.xA, sp.offA), pc(sp.vA, sp.xA, sp.offA), pe(sp.vB, sp.xB, sp.offB), pc(sp.vB, sp.xB, sp.offB),
                      pe(sp.vC, 0, sp.offC), pc(sp.vC, 0, sp.offC), ring, st, x);
      else
        launch_reduce(sp, n, pe(sp.vA, sp.xA, sp.offA), pc(sp.vA, sp.xA, sp.offA), pe(sp.vB, sp.xB, sp.offB), pc(sp.vB, sp.xB, sp.offB),
                      pe(sp.vC, 0, sp.offC), pc(sp.vC, 0, sp.offC), ring, st, x);
      n_launches++;
    }
  }

  int run_ring(int ring, int32_t *d_energy, uint64_t *d_count, uint32_t *d_mod) {
    const Plan &pl = lp->plan;
    const bool first_ring = ring == RING_U64 || ring == RING_NONE;
    const int kind = P->kind;
    int32_t *ve = (int32_t *)var_e.p, *ie = (int32_t *)inv_e.p;
    char *vc = (char *)var_c.p, *ic = (char *)inv_c.p;
    const size_t csz = ring_count_bytes(ring);
    const InputRec *d_in = (const InputRec *)inputs.p;
    const int32_t *d_l = (const int32_t *)lists.p;
    int32_t *oe = (int32_t *)off_e.p; char *oc = (char *)off_c.p;
    // slot 0: (.) of the scalar inputs of the run-once segments; slot 1: scratch; slots 2 ..: one per branch in flight
    launch_construct(kind, d_in, nullptr, 0, nullptr, 0, d_l + gsc_at, n_gsc, nullptr, 0, 1, ve, vc, ie, ic, oe, oc, ring, st);
    n_launches++;
    for (size_t si = 0; si < lp->segs.size(); si++) {
      const LocalSeg &s = lp->segs[si];
      const int f = (int)s.fixed.size();
      if (f == 0) {
        launch_construct(kind, d_in, nullptr, 0, d_l + inv_at[si], (int)s.list_inv.size(), nullptr, 0, nullptr, 0, 1, ve, vc, ie, ic,
                         oe + 1, oc + csz, ring, st);
        n_launches += 2;
        launch_steps(s, 1, nullptr, ring);
        if (first_ring) { fma_done += s.fma; bytes_done += s.bytes; n_sequences++; }
        continue;
      }
      // ---- a sliced segment: enumerate the assignments of F, prune, contract the survivors in batches, (+)-accumulate
      std::vector<std::pair<int, int>> adj_pairs;            // MIS: positions in F of adjacent fixed vertices
      if (kind == BBTN_MIS) {
        std::vector<int> posF(P->n, -1);
        for (int j = 0; j < f; j++) posF[s.fixed[j]] = j;
        for (int e = 0; e < P->m; e++) if (posF[P->eu[e]] >= 0 && posF[P->ev[e]] >= 0) adj_pairs.push_back({posF[P->eu[e]], posF[P->ev[e]]});
      }
      const uint32_t n_x = 1u << f;
      const uint32_t chunk = std::min<uint32_t>(n_x, 1u << 14);
      bool first = true;
      std::vector<uint8_t> live;                              // rows of the branches that survived pruning, not yet contracted
      auto flush = [&](bool all) -> int {                     // contract the survivors, nb_max at a time
        const int64_t n_live = (int64_t)live.size() / f;
        int64_t done = 0;
        while (n_live - done >= (all ? 1 : nb_max)) {
          const int64_t nb = std::min<int64_t>(nb_max, n_live - done);
          CUDA_TRY(h, assign.ensure((size_t)nb_max * f));
          CUDA_TRY(h, cudaMemcpyAsync(assign.p, live.data() + (size_t)done * f, (size_t)nb * f, cudaMemcpyHostToDevice, st));
          const uint8_t *xs = (const uint8_t *)assign.p;
          launch_construct(kind, d_in, d_l + var_at[si], (int)s.list_var.size(), d_l + inv_at[si], (int)s.list_inv.size(),
                           d_l + sc_at[si], (int)s.list_scalar.size(), xs, f, nb, ve, vc, ie, ic, oe + 2, oc + 2 * csz, ring, st);
          launch_steps(s, nb, xs, ring);
          launch_accumulate((int64_t)1 << s.acc_rank, nb, ve + s.tmp_off * nb, vc + (size_t)s.tmp_off * nb * csz, oe + 2, oc + 2 * csz,
                            ie + s.acc_off, ic + (size_t)s.acc_off * csz, first ? 1 : 0, ring, st);
          CUDA_TRY(h, cudaStreamSynchronize(st));             // the staging rows are reused by the next batch
          n_launches += 4;
          first = false;
          done += nb;
          if (first_ring) { n_contracted += nb; n_sequences++; fma_done += (double)nb * s.fma; bytes_done += (double)nb * s.bytes; }
        }
        live.erase(live.begin(), live.begin() + (size_t)done * f);
        return BBTN_OK;
      };
      for (uint32_t x0 = 0; x0 < n_x; x0 += chunk) {
        std::vector<uint8_t> rows((size_t)chunk * f);
        for (uint32_t i = 0; i < chunk; i++) for (int j = 0; j < f; j++) rows[(size_t)i * f + j] = (uint8_t)(((x0 + i) >> j) & 1u);
        std::vector<char> skip(chunk, 0);
        for (uint32_t i = 0; i < chunk; i++)
          for (auto &pr : adj_pairs) if ((((x0 + i) >> pr.first) & 1u) && (((x0 + i) >> pr.second) & 1u)) { skip[i] = 1; break; }
        if (first_ring) for (uint32_t i = 0; i < chunk; i++) n_infeasible += skip[i];
        if (have_inc && n_regions > 0) {
          // global pruning: a branch whose bound is strictly worse than the incumbent holds no optimum
          std::vector<int32_t> bound(chunk);
          int rc = bbtn_region_bound(h, roff, rv, n_regions, s.fixed.data(), f, rows.data(), chunk, bound.data(), st);
          if (rc) return rc;
          for (uint32_t i = 0; i < chunk; i++) {
            if (skip[i]) continue;
            const bool worse = kind == BBTN_ISING ? bound[i] > inc : bound[i] < inc;
            if (bound[i] == BBTN_NEG_INF || worse) { skip[i] = 1; if (first_ring) n_pruned++; }
          }
        }
        for (uint32_t i = 0; i < chunk; i++)
          if (!skip[i]) live.insert(live.end(), rows.begin() + (size_t)i * f, rows.begin() + (size_t)(i + 1) * f);
        int rc = flush(x0 + chunk >= n_x);
        if (rc) return rc;
      }
      if (first) {                                            // every branch pruned: the boundary tensor is the zero tensor
        launch_accumulate((int64_t)1 << s.acc_rank, 0, nullptr, nullptr, nullptr, nullptr, ie + s.acc_off, ic + (size_t)s.acc_off * csz, 1, ring, st);
        n_launches++;
      }
    }
    const bool has_root = pl.result_offset >= 0;
    launch_finalize(kind, 1, has_root ? ie + pl.result_offset : nullptr, has_root ? ic + (size_t)pl.result_offset * csz : nullptr, 0,
                    oe, oc, d_energy, d_count, d_mod, ring, st);
    n_launches++;
    CUDA_TRY(h, cudaGetLastError());
    return BBTN_OK;
  }
};

// run fn(i) for i in [0, n) on the host's cores (planning candidates are independent of one another)
template <class F> void parallel_for(size_t n, F fn) {
  const size_t nt = std::min<size_t>(n, std::max(1u, std::thread::hardware_concurrency()));
  if (nt <= 1) { for (size_t i = 0; i < n; i++) fn(i); return; }
  std::atomic<size_t> next{0};
  std::vector<std::thread> th;
  for (size_t t = 0; t < nt; t++) th.emplace_back([&] { for (size_t i; (i = next.fetch_add(1)) < n;) fn(i); });
  for (auto &t : th) t.join();
}

// Candidate trees: the caller's tree if there is one; else elimination trees along the vertex-id order, the
// min-degree order and nested-min-cut sweeps with several look-ahead windows (plan.cpp).  The driver plans
// every candidate and keeps the cheapest one that fits.
void candidate_trees(bbtn_handle *h, std::vector<std::unique_ptr<Problem>> &out, const std::vector<int> &deltas, bool plain_orders) {
  const Problem &P0 = h->P;
  if (!P0.tree_l.empty() || P0.n + P0.m <= 1) { out.push_back(std::make_unique<Problem>(P0)); return; }
  std::vector<std::vector<int>> orders;
  std::vector<int> natural(P0.n);
  for (int v = 0; v < P0.n; v++) natural[v] = v;
  if (plain_orders) { orders.push_back(natural); orders.push_back(min_degree_order(P0, {})); }
  int w0 = 0; double c0 = 0;
  { std::vector<int32_t> l, r; elimination_tree_for_order(P0, {}, natural, l, r, w0, c0); }
  // base orders of the nested-min-cut sweeps: the vertex ids, the caller's hints (bbtn_add_sweep_order), and each reversed
  std::vector<std::vector<int>> bases;
  bases.push_back(natural);
  for (auto &o : h->sweep_orders) bases.push_back(o);
  const size_t nb0 = bases.size();
  for (size_t i = 0; i < nb0; i++) bases.push_back(std::vector<int>(bases[i].rbegin(), bases[i].rend()));
  struct Job { size_t base; int half, delta; };
  std::vector<Job> jobs;
  std::vector<int> widths(bases.size(), w0);
  if (plain_orders) for (size_t i = 1; i < bases.size(); i++) orders.push_back(bases[i]);
  parallel_for(bases.size(), [&](size_t i) {                            // the look-ahead windows scale with each sweep's width
    if (i == 0) return;
    std::vector<int32_t> l, r; double c = 0;
    elimination_tree_for_order(P0, {}, bases[i], l, r, widths[i], c);
  });
  for (size_t i = 0; i < bases.size(); i++)
    for (int delta : deltas)
      for (int half : {4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14, 16}) jobs.push_back({i, half, delta});   // windows of 2 .. 8 sweep widths
  const size_t first_job = orders.size();
  orders.resize(first_job + jobs.size());
  parallel_for(jobs.size(), [&](size_t j) {
    orders[first_job + j] = mincut_sweep_order(P0, jobs[j].delta, std::max(8, jobs[j].half * widths[jobs[j].base] / 2), &bases[jobs[j].base]);
  });
  out.resize(orders.size());
  parallel_for(orders.size(), [&](size_t i) {
    auto P = std::make_unique<Problem>(P0);
    int w = 0; double c = 0;
    elimination_tree_for_order(P0, {}, orders[i], P->tree_l, P->tree_r, w, c);
    out[i] = std::move(P);
  });
}

void write_plan_stats(const LocalPlan &lp, int64_t *stats, double *work, bool search) {
  if (stats) {
    std::memset(stats, 0, 12 * sizeof(int64_t));
    stats[0] = (int64_t)lp.segs.size(); stats[1] = lp.n_sliced_segs;
    stats[2] = lp.n_slices > 9e18 ? INT64_MAX : (int64_t)lp.n_slices;
    stats[6] = lp.max_fixed; stats[7] = lp.plan.max_rank;
    stats[8] = (lp.plan.arena_invariant_elems + lp.plan.arena_variant_elems) * (search ? 4 : 12);      // with one branch in flight
  }
  if (work) { work[0] = lp.fma_total; work[1] = lp.bytes_total / (search ? 3.0 : 1.0); work[2] = work[3] = 0; }
}

// plan at log2_target, lowering the threshold while no candidate's arena fits the memory budget; among the
// candidates that fit, the one that moves the fewest bytes
int plan_within_budget(bbtn_handle *h, int32_t log2_target, int64_t budget, LocalPlan &lp, std::shared_ptr<Problem> &P_out) {
  const int64_t per_elem = (h->P.flags & BBTN_SEARCH_ONLY) ? 4 : 12;
  if (h->local_choice && h->local_choice->log2_target == log2_target && h->local_choice->n_hints == h->sweep_orders.size() &&
      (h->local_choice->budget == budget ||
       (budget > 0 && (h->local_choice->lp.plan.arena_invariant_elems + h->local_choice->lp.plan.arena_variant_elems) * per_elem <= budget &&
        h->local_choice->lp.cap_rank == log2_target))) {
    lp = h->local_choice->lp; P_out = h->local_choice->P;       // same request (or an unconstrained choice that also fits this budget)
    return BBTN_OK;
  }
  std::vector<std::unique_ptr<Problem>> cands;
  candidate_trees(h, cands, {4}, true);
  bool widened = !h->P.tree_l.empty();                        // a caller's tree is the only candidate
  std::string last_err; int last_rc = BBTN_ESHAPE;
  for (int cap = log2_target; cap >= 1; cap--) {
    std::vector<LocalPlan> plans(cands.size());
    std::vector<int> rcs(cands.size(), 0);
    std::vector<std::string> errs(cands.size());
    parallel_for(cands.size(), [&](size_t i) { rcs[i] = make_local_plan(*cands[i], cap, plans[i], errs[i]); });
    int best = -1;
    for (size_t i = 0; i < cands.size(); i++) {
      if (rcs[i]) { last_rc = rcs[i]; last_err = errs[i]; continue; }
      if (budget > 0 && (plans[i].plan.arena_invariant_elems + plans[i].plan.arena_variant_elems) * per_elem > budget) { last_rc = BBTN_ENOMEM; last_err = "arena does not fit the device-memory budget"; continue; }
      if (best < 0 || plans[i].bytes_total < plans[best].bytes_total) best = (int)i;
    }
    if (best >= 0 && !widened && plans[best].bytes_total > 1e14) {
      // an expensive plan (seconds of streaming): the cost of a plan is erratic in the details of the sweep, so it pays to
      // look at more of them -- the same bases and windows with other round sizes of the min-cut sweep
      widened = true;
      std::vector<std::unique_ptr<Problem>> more;
      candidate_trees(h, more, {2, 8, 16}, false);
      std::vector<LocalPlan> plans2(more.size());
      std::vector<int> rc2(more.size(), 0);
      std::vector<std::string> err2(more.size());
      parallel_for(more.size(), [&](size_t i) { rc2[i] = make_local_plan(*more[i], cap, plans2[i], err2[i]); });
      int b2 = -1;
      for (size_t i = 0; i < more.size(); i++) {
        if (rc2[i] || (budget > 0 && (plans2[i].plan.arena_invariant_elems + plans2[i].plan.arena_variant_elems) * per_elem > budget)) continue;
        if (plans2[i].bytes_total < plans[best].bytes_total && (b2 < 0 || plans2[i].bytes_total < plans2[b2].bytes_total)) b2 = (int)i;
      }
      if (b2 >= 0) { plans[best] = std::move(plans2[b2]); cands[best] = std::move(more[b2]); }
      for (auto &m : more) if (m) cands.push_back(std::move(m));     // keep them for lower thresholds, should this one not be final
    }
    if (best >= 0) {
      lp = std::move(plans[best]); P_out = std::move(cands[best]);
      h->local_choice = std::make_unique<bbtn_handle::LocalChoice>();
      h->local_choice->log2_target = log2_target; h->local_choice->budget = budget; h->local_choice->n_hints = h->sweep_orders.size();
      h->local_choice->lp = lp; h->local_choice->P = P_out;
      return BBTN_OK;
    }
  }
  return fail(h, last_rc, last_err);
}

}  // namespace

extern "C" {

int bbtn_add_sweep_order(bbtn_handle *h, const int32_t *order) {
  if (!h || !order) return fail(h, BBTN_EINVAL, "null argument");
  std::vector<int> o(order, order + h->P.n);
  std::vector<char> seen(h->P.n, 0);
  for (int v : o) {
    if (v < 0 || v >= h->P.n || seen[v]) return fail(h, BBTN_EINVAL, "order is not a permutation of the vertices");
    seen[v] = 1;
  }
  h->sweep_orders.push_back(std::move(o));
  return BBTN_OK;
}

int bbtn_local_plan_query(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes, int64_t *stats, double *work) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  if (log2_target < 1 || log2_target > 32) return fail(h, BBTN_EINVAL, "log2_target must be in 1..32");
  LocalPlan lp; std::shared_ptr<Problem> P;
  int rc = plan_within_budget(h, log2_target, mem_budget_bytes, lp, P);
  if (rc) return rc;
  write_plan_stats(lp, stats, work, (h->P.flags & BBTN_SEARCH_ONLY) != 0);
  return BBTN_OK;
}

int bbtn_solve_local(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes,
                     const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions, int32_t incumbent_hint,
                     int32_t *energy, uint64_t *count, uint32_t *count_mod, int64_t *stats, double *work, void *stream) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  if (!energy || !count || n_regions < 0 || (n_regions > 0 && (!region_offsets || !region_vertices)))
    return fail(h, BBTN_EINVAL, "bad solve_local arguments");
  if (log2_target < 1 || log2_target > 32) return fail(h, BBTN_EINVAL, "log2_target must be in 1..32");
  if (h->P.flags & BBTN_IO_DEVICE) return fail(h, BBTN_EINVAL, "bbtn_solve_local needs a host-pointer handle");
  const bool crt = (h->P.flags & BBTN_COUNT_CRT) != 0;
  if (count_mod && !crt) return fail(h, BBTN_EINVAL, "count_mod needs a handle built with BBTN_COUNT_CRT");
  if (!have_device()) return fail(h, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  if (mem_budget_bytes <= 0) {
    size_t free_b = 0, total_b = 0;
    CUDA_TRY(h, cudaMemGetInfo(&free_b, &total_b));
    mem_budget_bytes = (int64_t)((double)free_b * 0.94);
  }
  LocalPlan lp; std::shared_ptr<Problem> Pt;
  int rc = plan_within_budget(h, log2_target, mem_budget_bytes, lp, Pt);
  if (rc) return rc;
  const Problem *P = Pt.get();
  LocalRun run{h, P, &lp, (cudaStream_t)stream};
  {
    // branches of a stretch that are small are contracted many at a time (the batch axis of the kernels): as many as fit
    // the budget next to the invariant arena, at most 1024 and never more than the largest stretch has
    const int64_t per_elem = (h->P.flags & BBTN_SEARCH_ONLY) ? 4 : 12;
    const int64_t inv_b = lp.plan.arena_invariant_elems * per_elem, var_b = std::max<int64_t>(lp.plan.arena_variant_elems * per_elem, 1);
    int64_t most = 1;
    for (const LocalSeg &sg : lp.segs) most = std::max<int64_t>(most, (int64_t)1 << std::min<size_t>(sg.fixed.size(), 20));
    run.nb_max = std::max<int64_t>(1, std::min<int64_t>({(mem_budget_bytes - inv_b) / var_b, (int64_t)1024, most}));
  }
  run.roff = region_offsets; run.rv = region_vertices; run.n_regions = n_regions;
  run.have_inc = incumbent_hint != BBTN_NEG_INF; run.inc = incumbent_hint;
  if ((rc = run.upload())) return rc;
  const bool search = (h->P.flags & BBTN_SEARCH_ONLY) != 0;
  // CRT mode: a second pass with both prime residues packed in one 64-bit count (the plan has streaming steps only)
  const int n_rings = search ? 1 : ((crt && count_mod) ? 2 : 1);
  const int rings[2] = {search ? (int)RING_NONE : (int)RING_U64, (int)RING_P12};
  for (int ring = 0; ring < n_rings; ring++)
    if ((rc = run.run_ring(rings[ring], (int32_t *)run.res_e.p, (uint64_t *)run.res_c.p, (uint32_t *)run.res_m.p))) return rc;
  int32_t e; uint64_t c; uint32_t cm[2] = {0, 0};
  CUDA_TRY(h, cudaMemcpyAsync(&e, run.res_e.p, 4, cudaMemcpyDeviceToHost, run.st));
  CUDA_TRY(h, cudaMemcpyAsync(&c, run.res_c.p, 8, cudaMemcpyDeviceToHost, run.st));
  if (n_rings == 2) CUDA_TRY(h, cudaMemcpyAsync(cm, run.res_m.p, 8, cudaMemcpyDeviceToHost, run.st));
  CUDA_TRY(h, cudaStreamSynchronize(run.st));
  *energy = e; *count = c;
  if (count_mod) { count_mod[0] = cm[0]; count_mod[1] = cm[1]; }
  write_plan_stats(lp, stats, work, (h->P.flags & BBTN_SEARCH_ONLY) != 0);
  if (stats) {
    stats[3] = run.n_contracted; stats[4] = run.n_infeasible; stats[5] = run.n_pruned; stats[9] = run.n_launches;
    stats[8] = (lp.plan.arena_invariant_elems + lp.plan.arena_variant_elems * run.nb_max) * (((h->P.flags & BBTN_SEARCH_ONLY) != 0) ? 4 : 12);
    stats[10] = run.nb_max; stats[11] = run.n_sequences;
  }
  if (work) { work[2] = run.fma_done; work[3] = run.bytes_done / (((h->P.flags & BBTN_SEARCH_ONLY) != 0) ? 3.0 : 1.0); }
  return BBTN_OK;
}

}  // extern "C"
