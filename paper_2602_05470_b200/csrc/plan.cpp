// plan.cpp -- host planner (see plan.h).  Plain C++17, no CUDA, no oracle code.
#include "plan.h"
#include <cmath>

#include <algorithm>
#include <map>
#include <set>

namespace bbtn {
namespace {

enum { ST_EINVAL = 1, ST_ESHAPE = 4 };

// First-fit free-list allocator over element offsets (sizes are powers of two).  Every block is a
// multiple of 4 elements, so every tensor starts 16-byte aligned in both planes (the vectorised kernels
// need that; a 2-element bond tensor in front of a 2^31-element one must not push it off alignment).
struct Arena {
  std::map<int64_t, int64_t> free_;   // offset -> size
  int64_t top = 0;                    // high-water mark
  static int64_t round4(int64_t n) { return (n + 3) & ~(int64_t)3; }
  int64_t alloc(int64_t n) {
    n = round4(n);
    for (auto it = free_.begin(); it != free_.end(); ++it) {
      if (it->second >= n) {
        int64_t off = it->first, rest = it->second - n;
        free_.erase(it);
        if (rest > 0) free_[off + n] = rest;
        return off;
      }
    }
    // grow: extend a trailing free block if there is one
    if (!free_.empty()) {
      auto last = std::prev(free_.end());
      if (last->first + last->second == top) {
        int64_t off = last->first;
        top = off + n;
        free_.erase(last);
        return off;
      }
    }
    int64_t off = top;
    top += n;
    return off;
  }
  void release(int64_t off, int64_t n) {
    n = round4(n);
    auto it = free_.emplace(off, n).first;
    auto nx = std::next(it);
    if (nx != free_.end() && it->first + it->second == nx->first) { it->second += nx->second; free_.erase(nx); }
    if (it != free_.begin()) {
      auto pv = std::prev(it);
      if (pv->first + pv->second == it->first) { pv->second += it->second; free_.erase(it); }
    }
  }
};

struct TRef {
  bool removed = true;            // folded into offset[b] / not yet produced
  bool variant = false;
  std::vector<int> idx;           // idx[p] = index label at bit p
  int64_t off = 0;
  std::map<int, int> sub;         // unfinished indices -> number of input tensors in the subtree carrying them
  int lc = 0;                     // every count of this tensor is <= 2^lc (inputs: 1; (.) adds, (+) over 2^k terms adds k)
};

int pos_of(const std::vector<int> &v, int x) {
  for (size_t i = 0; i < v.size(); i++) if (v[i] == x) return (int)i;
  return -1;
}

}  // namespace

void derive_tree(const Problem &P, const std::vector<int32_t> &fixed,
                 std::vector<int32_t> &tl, std::vector<int32_t> &tr) {
  const int n = P.n, m = P.m, n_in = n + m;
  std::vector<char> isfixed(n, 0);
  for (int v : fixed) isfixed[v] = 1;
  // --- greedy min-degree (ties: min fill, then lowest id) elimination order on the free vertices
  std::vector<std::set<int>> adj(n);
  for (int e = 0; e < m; e++) {
    int u = P.eu[e], v = P.ev[e];
    if (isfixed[u] || isfixed[v]) continue;
    adj[u].insert(v); adj[v].insert(u);
  }
  std::vector<char> done(n, 0);
  std::vector<int> order;
  int n_free = 0;
  for (int v = 0; v < n; v++) if (!isfixed[v]) n_free++;
  for (int it = 0; it < n_free; it++) {
    int best = -1; size_t bd = 0; long bf = 0;
    for (int v = 0; v < n; v++) {
      if (isfixed[v] || done[v]) continue;
      size_t d = adj[v].size();
      if (best >= 0 && d > bd) continue;
      long fill = 0;
      if (d <= 12) {
        for (auto a = adj[v].begin(); a != adj[v].end(); ++a)
          for (auto b = std::next(a); b != adj[v].end(); ++b)
            if (!adj[*a].count(*b)) fill++;
      }
      if (best < 0 || d < bd || (d == bd && fill < bf)) { best = v; bd = d; bf = fill; }
    }
    order.push_back(best);
    done[best] = 1;
    std::vector<int> nb(adj[best].begin(), adj[best].end());
    for (int a : nb) adj[a].erase(best);
    for (size_t i = 0; i < nb.size(); i++)
      for (size_t j = i + 1; j < nb.size(); j++) { adj[nb[i]].insert(nb[j]); adj[nb[j]].insert(nb[i]); }
    adj[best].clear();
  }
  // --- bucket elimination along an order: merge all live tensors carrying v, smallest first.
  //     Returns (width = largest merged label set, cost = sum of 2^|union| over the merges).
  auto eliminate = [&](const std::vector<int> &ord, std::vector<int32_t> &ol, std::vector<int32_t> &orr, int &width, double &cost) {
    std::map<int, std::set<int>> live;            // tensor id -> labels
    std::vector<std::set<int>> occ(n);            // label -> tensor ids
    for (int t = 0; t < n_in; t++) {
      std::set<int> s;
      if (t < m) { if (!isfixed[P.eu[t]]) s.insert(P.eu[t]); if (!isfixed[P.ev[t]]) s.insert(P.ev[t]); }
      else if (!isfixed[t - m]) s.insert(t - m);
      for (int i : s) occ[i].insert(t);
      live[t] = s;
    }
    int nxt = n_in;
    ol.clear(); orr.clear(); width = 0; cost = 0;
    auto merge = [&](int a, int b) {
      std::set<int> sa = live[a], sb = live[b];
      live.erase(a); live.erase(b);
      for (int i : sa) occ[i].erase(a);
      for (int i : sb) occ[i].erase(b);
      std::set<int> uni = sa;
      uni.insert(sb.begin(), sb.end());
      width = std::max(width, (int)uni.size());
      cost += std::ldexp(1.0, (int)uni.size());
      std::set<int> keep;
      for (int i : uni) if (!occ[i].empty()) keep.insert(i);   // still carried by another live tensor
      for (int i : keep) occ[i].insert(nxt);
      live[nxt] = keep;
      ol.push_back(a); orr.push_back(b);
      return nxt++;
    };
    for (int v : ord) {
      while (occ[v].size() >= 2) {
        int a = -1, b = -1;
        for (int t : occ[v]) {
          if (a < 0 || live[t].size() < live[a].size()) { b = a; a = t; }
          else if (b < 0 || live[t].size() < live[b].size()) b = t;
        }
        merge(a, b);
      }
    }
    std::vector<std::pair<size_t, int>> rest;
    for (auto &kv : live) rest.push_back({kv.second.size(), kv.first});
    std::sort(rest.begin(), rest.end());
    if (!rest.empty()) {
      int cur = rest[0].second;
      for (size_t i = 1; i < rest.size(); i++) cur = merge(cur, rest[i].second);
    }
  };
  // candidates: the min-degree order and the plain vertex-id order (a frontier sweep for instances
  // numbered row-major, e.g. lattices and King's subgraphs); keep the narrower, then the cheaper one
  std::vector<int> natural;
  for (int v = 0; v < n; v++) if (!isfixed[v]) natural.push_back(v);
  std::vector<int32_t> l2, r2;
  int w1 = 0, w2 = 0; double c1 = 0, c2 = 0;
  eliminate(order, tl, tr, w1, c1);
  eliminate(natural, l2, r2, w2, c2);
  if (w2 < w1 || (w2 == w1 && c2 < c1)) { tl.swap(l2); tr.swap(r2); }
}

int make_plan(const Problem &P, const std::vector<int32_t> &fixed, int force_mode, bool enforce_cap,
              Plan &out, std::string &err, bool single_arena, bool want_labels) {
  const int n = P.n, m = P.m, n_in = n + m;
  out = Plan();
  out.fixed = fixed;
  std::vector<int> fpos(n, -1);
  for (size_t j = 0; j < fixed.size(); j++) {
    int v = fixed[j];
    if (v < 0 || v >= n) { err = "fixed vertex id out of range"; return ST_EINVAL; }
    if (fpos[v] >= 0) { err = "duplicate fixed vertex"; return ST_EINVAL; }
    fpos[v] = (int)j;
  }
  int cap_rank = 0;
  while (((int64_t)1 << (cap_rank + 1)) <= P.max_elements && cap_rank < 32) cap_rank++;

  // ---- inputs
  std::vector<int> occ_total(n, 0);
  for (int e = 0; e < m; e++) { if (fpos[P.eu[e]] < 0) occ_total[P.eu[e]]++; if (fpos[P.ev[e]] < 0) occ_total[P.ev[e]]++; }
  for (int i = 0; i < n; i++) if (fpos[i] < 0) occ_total[i]++;
  Arena av, ai;
  std::vector<TRef> T((size_t)n_in);
  out.inputs.resize((size_t)n_in);
  for (int t = 0; t < n_in; t++) {
    InputRec &r = out.inputs[t];
    r.type = t < m ? 0 : 1;
    r.u = t < m ? P.eu[t] : t - m;
    r.v = t < m ? P.ev[t] : -1;
    r.w = t < m ? P.ew[t] : P.vw[t - m];
    r.fu = fpos[r.u];
    r.fv = r.v >= 0 ? fpos[r.v] : -1;
    r.su = (r.fu < 0 && occ_total[r.u] == 1) ? 1 : 0;
    r.sv = (r.v >= 0 && r.fv < 0 && occ_total[r.v] == 1) ? 1 : 0;
    r.bu = r.bv = -1;
    int rank = 0;
    TRef &x = T[t];
    x.idx.clear();
    if (r.fu < 0 && !r.su) { r.bu = rank++; x.idx.push_back(r.u); x.sub[r.u] = 1; }
    if (r.v >= 0 && r.fv < 0 && !r.sv) { r.bv = rank++; x.idx.push_back(r.v); x.sub[r.v] = 1; }
    r.rank = rank;
    x.lc = r.su + r.sv;             // K1 pre-sums single-owner indices: up to 2 (4) unit counts added
    r.variant = (single_arena || r.fu >= 0 || r.fv >= 0) ? 1 : 0;
    r.offset = -1;
    if (rank == 0) { out.scalar_inputs.push_back(t); x.removed = true; continue; }
    x.removed = false;
    x.variant = r.variant != 0;
    x.off = (x.variant ? av : ai).alloc((int64_t)1 << rank);
    r.offset = x.off;
  }

  // ---- tree
  std::vector<int32_t> tl = P.tree_l, tr = P.tree_r;
  if (tl.empty() && n_in > 1) derive_tree(P, fixed, tl, tr);
  if ((int)tl.size() != n_in - 1) { err = "contraction tree must have n_inputs - 1 steps"; return ST_EINVAL; }
  T.resize((size_t)(n_in + tl.size()));
  std::vector<char> used(T.size(), 0);

  auto release = [&](TRef &x) { (x.variant ? av : ai).release(x.off, (int64_t)1 << x.idx.size()); };

  for (size_t s = 0; s < tl.size(); s++) {
    int Li = tl[s], Ri = tr[s], Oi = n_in + (int)s;
    if (Li < 0 || Ri < 0 || Li >= Oi || Ri >= Oi || Li == Ri || used[Li] || used[Ri]) {
      err = "malformed contraction tree (step " + std::to_string(s) + ")"; return ST_EINVAL;
    }
    used[Li] = used[Ri] = 1;
    TRef &L = T[Li], &R = T[Ri], &O = T[Oi];
    if (L.removed && R.removed) { O.removed = true; continue; }
    if (L.removed || R.removed) { O = L.removed ? R : L; continue; }   // scalar operand lives in offset[b]
    // merged occurrence counts -> I_O = labels still carried by an input outside this subtree
    O.removed = false;
    O.variant = L.variant || R.variant;
    const int lc_in = std::max(L.lc, R.lc), lc_sum = L.lc + R.lc;
    O.sub = L.sub;
    for (auto &kv : R.sub) O.sub[kv.first] += kv.second;
    for (auto it = O.sub.begin(); it != O.sub.end();) {
      if (it->second >= occ_total[it->first]) it = O.sub.erase(it); else ++it;
    }
    auto inO = [&](int lab) { return O.sub.count(lab) != 0; };
    // the larger operand streams in its own layout ("A"), the smaller one is gathered ("B")
    const bool swap = R.idx.size() > L.idx.size();
    TRef &A = swap ? R : L, &B = swap ? L : R;
    std::vector<int> gl, kl, ml, nl;     // labels per class, in A's bit order (N: B's order)
    for (int lab : A.idx) {
      bool inB = pos_of(B.idx, lab) >= 0;
      if (inB && inO(lab)) gl.push_back(lab);
      else if (inB) kl.push_back(lab);
      else if (inO(lab)) ml.push_back(lab);
      else { err = "internal: index summed too late"; return ST_EINVAL; }
    }
    for (int lab : B.idx) {
      if (pos_of(A.idx, lab) >= 0) continue;
      if (!inO(lab)) { err = "internal: index summed too late"; return ST_EINVAL; }
      nl.push_back(lab);
    }
    const int rA = (int)A.idx.size(), rB = (int)B.idx.size();
    const int lg = (int)gl.size(), lk = (int)kl.size(), lm = (int)ml.size(), ln = (int)nl.size();
    const int rO = lg + lm + ln;
    out.rho += std::max(0, rO - cap_rank);                     // Eq. 4, T_target = 2^cap_rank
    if (enforce_cap && (rO > cap_rank || rA > cap_rank)) {
      err = "intermediate of rank " + std::to_string(std::max(rO, rA)) + " exceeds max_elements_per_leaf";
      return ST_ESHAPE;
    }
    out.max_rank = std::max(out.max_rank, std::max(rO, std::max(rA, rB)));
    if (want_labels) {
      std::vector<int32_t> labs;
      for (int lab : gl) labs.push_back(lab);
      for (int lab : ml) labs.push_back(lab);
      for (int lab : nl) labs.push_back(lab);
      out.node_labels.push_back(std::move(labs));
    }
    const bool var = O.variant;
    Arena &ao = var ? av : ai;
    const double fma = (double)((int64_t)1 << (rO + lk));
    bool tiled = false;
    if (force_mode == 2) tiled = lk >= 1;
    else if (force_mode == 0) tiled = lk >= 4 && lm >= 5 && ln >= 5;
    O.lc = std::min(lc_sum + lk, 1 << 20);
    out.n_nodes++;
    if (var) out.n_variant_nodes++;
    (var ? out.fma_variant : out.fma_invariant) += fma;

    if (!tiled) {
      Step st;
      // few outputs and a long sum: one CTA per output ((+)-reduction across the block); everything else streams
      st.kind = (lk >= 8 && rO <= 10) ? STEP_REDUCE : STEP_ABSORB;
      st.variant = var;
      st.rO = rO; st.nK = lk;
      // output layout: A's surviving bits in A's order, then B's new bits
      O.idx.clear();
      for (int lab : A.idx) if (inO(lab)) O.idx.push_back(lab);
      for (int lab : nl) O.idx.push_back(lab);
      for (int p = 0; p < rO; p++) {
        int pa = pos_of(A.idx, O.idx[p]), pb = pos_of(B.idx, O.idx[p]);
        st.addA[p] = pa >= 0 ? (1u << pa) : 0u;
        st.addB[p] = pb >= 0 ? (1u << pb) : 0u;
      }
      for (int j = 0; j < lk; j++) {
        st.kA[j] = 1u << pos_of(A.idx, kl[j]);
        st.kB[j] = 1u << pos_of(B.idx, kl[j]);
      }
      O.off = ao.alloc((int64_t)1 << rO);
      st.offA = A.off; st.offB = B.off; st.offC = O.off;
      st.vA = A.variant; st.vB = B.variant; st.vC = var;
      st.rA = rA; st.rB = rB;
      st.fma = fma;
      st.bytes = 12.0 * ((double)((int64_t)1 << rA) + (double)((int64_t)1 << rB) + (double)((int64_t)1 << rO));
      (var ? out.bytes_variant : out.bytes_invariant) += st.bytes;
      out.steps.push_back(st);
      release(A); release(B);
    } else {
      // canonical GEMM order: A -> [g][k][m] (m fastest), B -> [g][k][n], C = [g][m][n]
      auto canon = [&](TRef &X, const std::vector<int> &freel, int64_t &off_out) -> bool {
        std::vector<int> want = freel;
        want.insert(want.end(), kl.begin(), kl.end());
        want.insert(want.end(), gl.begin(), gl.end());
        if (want == X.idx) { off_out = X.off; return false; }
        Step ps;
        ps.kind = STEP_PERMUTE; ps.variant = X.variant; ps.rO = (int)X.idx.size();
        for (size_t j = 0; j < want.size(); j++) ps.perm[j] = pos_of(X.idx, want[j]);
        Arena &ax = X.variant ? av : ai;
        off_out = ax.alloc((int64_t)1 << X.idx.size());
        ps.offA = X.off; ps.offC = off_out; ps.vA = ps.vC = X.variant; ps.rA = ps.rO;
        ps.bytes = 24.0 * (double)((int64_t)1 << X.idx.size());
        (X.variant ? out.bytes_variant : out.bytes_invariant) += ps.bytes;
        out.steps.push_back(ps);
        return true;
      };
      int64_t offA2, offB2;
      bool tmpA = canon(A, ml, offA2);
      bool tmpB = canon(B, nl, offB2);
      if (tmpA) release(A);          // the permuted copy replaces the original
      if (tmpB) release(B);
      Step st;
      st.kind = STEP_GEMM; st.variant = var;
      st.count_bits = std::min(lc_in + 1, 64);
      st.lg = lg; st.lm = lm; st.ln = ln; st.lk = lk; st.rO = rO; st.nK = lk;
      O.idx = nl;
      O.idx.insert(O.idx.end(), ml.begin(), ml.end());
      O.idx.insert(O.idx.end(), gl.begin(), gl.end());
      O.off = ao.alloc((int64_t)1 << rO);
      st.offA = offA2; st.offB = offB2; st.offC = O.off;
      st.vA = A.variant; st.vB = B.variant; st.vC = var;
      st.rA = rA; st.rB = rB;
      st.fma = fma;
      st.bytes = 12.0 * ((double)((int64_t)1 << rA) + (double)((int64_t)1 << rB) + (double)((int64_t)1 << rO));
      (var ? out.bytes_variant : out.bytes_invariant) += st.bytes;
      out.steps.push_back(st);
      (A.variant ? av : ai).release(offA2, (int64_t)1 << rA);
      (B.variant ? av : ai).release(offB2, (int64_t)1 << rB);
    }
  }
  for (size_t t = 0; t + 1 < T.size(); t++)
    if (!used[t]) { err = "contraction tree does not consume every tensor"; return ST_EINVAL; }
  TRef &root = T.back();
  if (!root.removed) {
    if (!root.idx.empty()) { err = "contraction tree root is not a scalar"; return ST_EINVAL; }
    out.result_offset = root.off;
    out.result_variant = root.variant;
  }
  out.arena_variant_elems = av.top;
  out.arena_invariant_elems = ai.top;
  return 0;
}

}  // namespace bbtn
