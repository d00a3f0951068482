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
  // a VIEW of a stored tensor with some of its indices fixed (local slicing): logical bit p lives at element
  // offset phys[p] (empty = dense, 1 << p); slice[j] = element stride of the j-th locally fixed index (0 if absent)
  bool ext = false;
  bool keep = false;              // read again by the next slice of a sliced segment: released when the segment ends
  std::vector<uint32_t> phys, slice;
};

int pos_of(const std::vector<int> &v, int x) {
  for (size_t i = 0; i < v.size(); i++) if (v[i] == x) return (int)i;
  return -1;
}

}  // namespace

// bucket elimination along an order of the free vertices: merge all live tensors carrying v, smallest first.
// Returns (width = largest merged label set, cost = sum of 2^|union| over the merges).
void elimination_tree_for_order(const Problem &P, const std::vector<int32_t> &fixed, const std::vector<int> &ord,
                                std::vector<int32_t> &ol, std::vector<int32_t> &orr, int &width, double &cost) {
  const int n = P.n, m = P.m, n_in = n + m;
  std::vector<char> isfixed(n, 0);
  for (int v : fixed) isfixed[v] = 1;
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
}

// greedy min-degree (ties: min fill, then lowest id) elimination order on the free vertices
std::vector<int> min_degree_order(const Problem &P, const std::vector<int32_t> &fixed) {
  const int n = P.n, m = P.m;
  std::vector<char> isfixed(n, 0);
  for (int v : fixed) isfixed[v] = 1;
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
  return order;
}

// Frontier sweep along nested minimum vertex cuts.  Starting from the vertex-id order (a row-major sweep for lattices
// and King's subgraphs), the eliminated set X grows in rounds: round k takes X u {the first k*delta vertices} as the
// source, everything beyond a window of `window` vertices as the sink, and a maximum flow with unit vertex capacities
// finds the smallest separator between them; X becomes the source side closest to the source.  On a King's subgraph
// at filling 0.8 the separators thread through the missing sites: ~30 kept sites where a straight row holds up to 39.
// The vertices a round adds are ordered greedily (the one that enlarges the frontier least goes first).
std::vector<int> mincut_sweep_order(const Problem &P, int delta, int window, const std::vector<int> *base) {
  const int n = P.n;
  // the sweep runs on POSITIONS of a base order (the vertex ids themselves when base == nullptr); mapped back at the end
  std::vector<int> posn(n);
  for (int i = 0; i < n; i++) posn[base ? (*base)[i] : i] = i;
  std::vector<std::vector<int>> adj(n);
  for (int e = 0; e < P.m; e++) { const int u = posn[P.eu[e]], v = posn[P.ev[e]]; adj[u].push_back(v); adj[v].push_back(u); }
  std::vector<char> inX(n, 0), front(n, 0);
  std::vector<int> order;
  order.reserve(n);
  auto add_slab = [&](std::vector<int> slab) {            // slab in id order
    std::vector<char> in_slab(n, 0);
    for (int v : slab) in_slab[v] = 1;
    size_t left = slab.size();
    while (left > 0) {
      int best = -1, bd = 0, bf = 0;
      for (int v : slab) {
        if (!in_slab[v]) continue;
        int newn = 0;
        for (int u : adj[v]) if (!inX[u] && !front[u] && u != v) newn++;
        const int d = newn - (front[v] ? 1 : 0), f = front[v] ? 0 : 1;
        if (best < 0 || d < bd || (d == bd && f < bf)) { best = v; bd = d; bf = f; }   // ties: lowest id (slab is sorted)
      }
      in_slab[best] = 0; left--;
      order.push_back(best); inX[best] = 1; front[best] = 0;
      for (int u : adj[best]) if (!inX[u]) front[u] = 1;
    }
  };
  int n_in_X = 0;
  for (int k = delta; n_in_X < n; k += delta) {
    const int lo = std::min(k, n), hi = std::min(n, k + window);
    std::vector<int> slab;
    if (hi >= n) {
      for (int v = 0; v < n; v++) if (!inX[v]) slab.push_back(v);
    } else {
      // role: 0 source (X or id < lo), 1 free, 2 sink (id >= hi and not in X)
      std::vector<int> idx(n, -1), free_v;
      for (int v = lo; v < hi; v++) if (!inX[v]) { idx[v] = (int)free_v.size(); free_v.push_back(v); }
      const int nF = (int)free_v.size(), S = 2 * nF, T = 2 * nF + 1;
      struct Edge { int to, cap; };
      std::vector<Edge> edges; std::vector<std::vector<int>> g((size_t)(2 * nF + 2));
      auto add = [&](int a, int b, int c) { g[a].push_back((int)edges.size()); edges.push_back({b, c}); g[b].push_back((int)edges.size()); edges.push_back({a, 0}); };
      const int INF = 1 << 29;
      for (int i = 0; i < nF; i++) {
        const int v = free_v[i];
        add(2 * i, 2 * i + 1, 1);
        bool s_adj = false, t_adj = false;
        for (int u : adj[v]) {
          if (idx[u] >= 0) add(2 * i + 1, 2 * idx[u], INF);
          else if (inX[u] || u < lo) s_adj = true;
          else t_adj = true;
        }
        if (s_adj) add(S, 2 * i, INF);
        if (t_adj) add(2 * i + 1, T, INF);
      }
      std::vector<int> par((size_t)(2 * nF + 2));
      while (true) {                                       // augmenting paths (the flow is at most a separator size)
        std::fill(par.begin(), par.end(), -2);
        par[S] = -1;
        std::vector<int> q{S};
        for (size_t h = 0; h < q.size() && par[T] == -2; h++)
          for (int ei : g[q[h]]) if (edges[ei].cap > 0 && par[edges[ei].to] == -2) { par[edges[ei].to] = ei; q.push_back(edges[ei].to); }
        if (par[T] == -2) break;
        for (int v = T; v != S;) { const int ei = par[v]; edges[ei].cap--; edges[ei ^ 1].cap++; v = edges[ei ^ 1].to; }
      }
      for (int v = 0; v < lo; v++) if (!inX[v]) slab.push_back(v);
      for (int i = 0; i < nF; i++) if (par[2 * i + 1] != -2) slab.push_back(free_v[i]);   // out-node reachable: source side
      std::sort(slab.begin(), slab.end());
    }
    n_in_X += (int)slab.size();
    add_slab(std::move(slab));
  }
  if (base) for (int &v : order) v = (*base)[v];
  return order;
}

void derive_tree(const Problem &P, const std::vector<int32_t> &fixed,
                 std::vector<int32_t> &tl, std::vector<int32_t> &tr) {
  // candidates: the min-degree order and the plain vertex-id order (a frontier sweep for instances
  // numbered row-major, e.g. lattices and King's subgraphs); keep the narrower, then the cheaper one
  std::vector<char> isfixed(P.n, 0);
  for (int v : fixed) isfixed[v] = 1;
  std::vector<int> natural;
  for (int v = 0; v < P.n; v++) if (!isfixed[v]) natural.push_back(v);
  std::vector<int32_t> l2, r2;
  int w1 = 0, w2 = 0; double c1 = 0, c2 = 0;
  elimination_tree_for_order(P, fixed, min_degree_order(P, fixed), tl, tr, w1, c1);
  elimination_tree_for_order(P, fixed, natural, l2, r2, w2, c2);
  if (w2 < w1 || (w2 == w1 && c2 < c1)) { tl.swap(l2); tr.swap(r2); }
}

namespace {

// ---------------------------------------------------------------------------------------------
// The planner proper: a step-by-step walk over the SSA tree.  make_plan() walks the whole tree under one
// fixed set; make_local_plan() walks it segment by segment, with a LOCAL fixed set inside the segments
// whose tensors would overflow T_target.
// ---------------------------------------------------------------------------------------------
struct Planner {
  const Problem &P;
  const int n, m, n_in;
  int force_mode; bool enforce_cap, single_arena, want_labels;
  int cap_rank = 0;
  Plan &out; std::string &err;
  std::vector<int> fpos;            // column of a fixed vertex inside `assign`, -1 when free
  std::vector<int> occ_total;       // number of input tensors carrying a (free) label
  Arena av, ai;
  std::vector<TRef> T;
  std::vector<char> used;
  std::vector<int32_t> tl, tr;
  // local planning: operands that must outlive the step (they are read again by the next slice)
  bool gather_friendly_b = false;                      // make_plan only: re-lay a mid-sized gathered operand (see do_step)
  struct Deferred { bool variant; int64_t off, ne; };
  std::vector<Deferred> deferred;                      // storage to give back when the sliced segment ends

  Planner(const Problem &P_, int force_mode_, bool enforce_cap_, bool single_arena_, bool want_labels_, Plan &out_, std::string &err_)
      : P(P_), n(P_.n), m(P_.m), n_in(P_.n + P_.m), force_mode(force_mode_), enforce_cap(enforce_cap_),
        single_arena(single_arena_), want_labels(want_labels_), out(out_), err(err_) {
    while (((int64_t)1 << (cap_rank + 1)) <= P.max_elements && cap_rank < 32) cap_rank++;
  }

  int set_fixed(const std::vector<int32_t> &fixed) {
    fpos.assign(n, -1);
    for (size_t j = 0; j < fixed.size(); j++) {
      int v = fixed[j];
      if (v < 0 || v >= n) { err = "fixed vertex id out of range"; return ST_EINVAL; }
      if (fpos[v] >= 0) { err = "duplicate fixed vertex"; return ST_EINVAL; }
      fpos[v] = (int)j;
    }
    return 0;
  }
  // occurrence counts under the CURRENT fixed set (call once for a whole-tree plan; the local planner calls it with
  // nothing fixed: labels outside a segment are not affected by the segment's slicing)
  void count_occurrences() {
    occ_total.assign(n, 0);
    for (int e = 0; e < m; e++) { if (fpos[P.eu[e]] < 0) occ_total[P.eu[e]]++; if (fpos[P.ev[e]] < 0) occ_total[P.ev[e]]++; }
    for (int i = 0; i < n; i++) if (fpos[i] < 0) occ_total[i]++;
  }
  int init_tree(const std::vector<int32_t> &fixed_for_tree) {
    out.inputs.resize((size_t)n_in);
    tl = P.tree_l; tr = P.tree_r;
    if (tl.empty() && n_in > 1) derive_tree(P, fixed_for_tree, tl, tr);
    if ((int)tl.size() != n_in - 1) { err = "contraction tree must have n_inputs - 1 steps"; return ST_EINVAL; }
    T.assign((size_t)(n_in + tl.size()), TRef());
    used.assign(T.size(), 0);
    return 0;
  }

  static uint32_t bit_of(const TRef &X, int pos) { return X.phys.empty() ? (pos < 32 ? (1u << pos) : 0u) : X.phys[pos]; }
  void release(TRef &x) {
    if (x.ext) return;                                  // a view: its storage belongs to the tensor it was cut from
    const int64_t ne = (int64_t)1 << x.idx.size();
    if (x.keep) deferred.push_back({x.variant, x.off, ne});
    else (x.variant ? av : ai).release(x.off, ne);
  }

  // input tensor t as K1 must build it under the current fixed set
  void add_input(int t) {
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
    x = TRef();
    if (r.fu < 0 && !r.su) { r.bu = rank++; x.idx.push_back(r.u); x.sub[r.u] = 1; }
    if (r.v >= 0 && r.fv < 0 && !r.sv) { r.bv = rank++; x.idx.push_back(r.v); x.sub[r.v] = 1; }
    r.rank = rank;
    x.lc = r.su + r.sv;             // K1 pre-sums single-owner indices: up to 2 (4) unit counts added
    r.variant = (single_arena || r.fu >= 0 || r.fv >= 0) ? 1 : 0;
    r.offset = -1;
    if (rank == 0) { x.removed = true; return; }
    x.removed = false;
    x.variant = r.variant != 0;
    x.off = (x.variant ? av : ai).alloc((int64_t)1 << rank);
    r.offset = x.off;
  }

  // plan tree step s; `launched` (optional) tells whether a device step was emitted
  int do_step(size_t s, bool *launched = nullptr) {
    if (launched) *launched = false;
    int Li = tl[s], Ri = tr[s], Oi = n_in + (int)s;
    if (Li < 0 || Ri < 0 || Li >= Oi || Ri >= Oi || Li == Ri || used[Li] || used[Ri]) {
      err = "malformed contraction tree (step " + std::to_string(s) + ")"; return ST_EINVAL;
    }
    used[Li] = used[Ri] = 1;
    TRef &L = T[Li], &R = T[Ri], &O = T[Oi];
    if (L.removed && R.removed) { O.removed = true; return 0; }
    if (L.removed || R.removed) { O = L.removed ? R : L; return 0; }   // scalar operand lives in offset[b]
    // merged occurrence counts -> I_O = labels still carried by an input outside this subtree
    O.removed = false;
    O.ext = false; O.keep = false; O.phys.clear(); O.slice.clear();
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
    if (!A.phys.empty() || !B.phys.empty()) tiled = false;     // views are not dense: only the streaming forms address them
    O.lc = std::min(lc_sum + lk, 1 << 20);
    out.n_nodes++;
    if (var) out.n_variant_nodes++;
    (var ? out.fma_variant : out.fma_invariant) += fma;
    if (launched) *launched = true;

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
      // The gathered operand is read at fb(o): its layout decides how many sectors a warp's loads touch.  A mid-sized B
      // (256+ elements) under a large output is first re-laid (K2) with its surviving indices in the ORDER OF THE OUTPUT
      // (then consecutive outputs read the same or consecutive elements) and the summed ones on top; without this the L1
      // data pipe, not HBM, bounds the write-heavy steps of balanced trees (7 sectors per load request on the cube).
      std::vector<int> b_idx = B.idx;
      int64_t b_off = B.off; bool b_tmp = false;
      if (gather_friendly_b && rO >= 16 && rB >= 8 && rB + 2 <= rO && B.phys.empty() && !B.ext && B.slice.empty() && rB <= 31) {
        std::vector<int> want;
        for (int lab : O.idx) if (pos_of(B.idx, lab) >= 0) want.push_back(lab);
        want.insert(want.end(), kl.begin(), kl.end());
        const size_t head = std::min<size_t>(want.size(), 7);
        if (!std::equal(want.begin(), want.begin() + head, B.idx.begin())) {
          Step ps;
          ps.kind = STEP_PERMUTE; ps.variant = B.variant; ps.rO = rB;
          for (size_t j = 0; j < want.size(); j++) ps.perm[j] = pos_of(B.idx, want[j]);
          b_off = (B.variant ? av : ai).alloc((int64_t)1 << rB);
          ps.offA = B.off; ps.offC = b_off; ps.vA = ps.vC = B.variant; ps.rA = ps.rO;
          ps.bytes = 24.0 * (double)((int64_t)1 << rB);
          (B.variant ? out.bytes_variant : out.bytes_invariant) += ps.bytes;
          out.steps.push_back(ps);
          b_idx = want; b_tmp = true;
        }
      }
      auto bit_b = [&](int pos) { return b_tmp ? (pos < 32 ? (1u << pos) : 0u) : bit_of(B, pos); };
      for (int p = 0; p < rO && p < 32; p++) {              // ranks above 32 occur only in dry runs (rho of an unsliced tree)
        int pa = pos_of(A.idx, O.idx[p]), pb = pos_of(b_idx, O.idx[p]);
        st.addA[p] = pa >= 0 ? bit_of(A, pa) : 0u;
        st.addB[p] = pb >= 0 ? bit_b(pb) : 0u;
      }
      for (int j = 0; j < lk && j < 32; j++) {
        st.kA[j] = bit_of(A, pos_of(A.idx, kl[j]));
        st.kB[j] = bit_b(pos_of(b_idx, kl[j]));
      }
      O.off = ao.alloc((int64_t)1 << rO);
      st.offA = A.off; st.offB = b_off; st.offC = O.off;
      st.vA = A.variant; st.vB = B.variant; st.vC = var;
      st.rA = rA; st.rB = rB;
      st.n_slice = (int32_t)std::max(A.slice.size(), B.slice.size());
      st.xA = A.ext ? 1 : 0; st.xB = B.ext ? 1 : 0;
      st.b_unit = B.lc == 0 ? 1 : 0;
      for (size_t j = 0; j < A.slice.size(); j++) st.sliceA[j] = A.slice[j];
      for (size_t j = 0; j < B.slice.size(); j++) st.sliceB[j] = B.slice[j];
      st.fma = fma;
      st.bytes = 12.0 * ((double)((int64_t)1 << rA) + (double)((int64_t)1 << rB) + (double)((int64_t)1 << rO));
      (var ? out.bytes_variant : out.bytes_invariant) += st.bytes;
      out.steps.push_back(st);
      if (b_tmp) (B.variant ? av : ai).release(b_off, (int64_t)1 << rB);      // the re-laid copy is scratch of this step
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
        for (size_t j = 0; j < want.size() && j < 32; j++) ps.perm[j] = pos_of(X.idx, want[j]);
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
      // a permuted copy is scratch of this step; an operand used in place follows the ordinary release rule
      if (tmpA) (A.variant ? av : ai).release(offA2, (int64_t)1 << rA); else release(A);
      if (tmpB) (B.variant ? av : ai).release(offB2, (int64_t)1 << rB); else release(B);
    }
    return 0;
  }

  int finish() {
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
};

}  // namespace

int make_plan(const Problem &P, const std::vector<int32_t> &fixed, int force_mode, bool enforce_cap,
              Plan &out, std::string &err, bool single_arena, bool want_labels) {
  out = Plan();
  out.fixed = fixed;
  Planner pl(P, force_mode, enforce_cap, single_arena, want_labels, out, err);
  pl.gather_friendly_b = force_mode != 2;                 // (the all-tiled test mode keeps its node kinds)
  int rc;
  if ((rc = pl.set_fixed(fixed))) return rc;
  pl.count_occurrences();
  if ((rc = pl.init_tree(fixed))) return rc;
  for (int t = 0; t < pl.n_in; t++) {
    pl.add_input(t);
    if (out.inputs[t].rank == 0) out.scalar_inputs.push_back(t);
  }
  for (size_t s = 0; s < pl.tl.size(); s++)
    if ((rc = pl.do_step(s))) return rc;
  return pl.finish();
}

// ---------------------------------------------------------------------------------------------
// make_local_plan (plan.h "local slicing")
// ---------------------------------------------------------------------------------------------
int make_local_plan(const Problem &P, int cap_rank, LocalPlan &out, std::string &err) {
  out = LocalPlan();
  out.cap_rank = cap_rank;
  const int n_in = P.n + P.m;
  if (P.tree_l.empty() && n_in > 1) { err = "make_local_plan needs a contraction tree"; return ST_EINVAL; }
  const int S = (int)P.tree_l.size(), n_t = n_in + S;

  // ---- pass 0: the unsliced structure (labels, liveness) from a dry walk
  std::vector<std::vector<int>> lab((size_t)n_t);
  std::vector<char> removed((size_t)n_t, 0);
  std::vector<int> alias((size_t)n_t, -1), cons((size_t)n_t, S);     // S = never consumed (the root)
  std::vector<int> sum_step(P.n, -1);
  {
    Plan dry; std::string e2;
    Planner pl(P, 1, false, true, false, dry, e2);
    pl.set_fixed({}); pl.count_occurrences();
    int rc = pl.init_tree({});
    if (rc) { err = e2; return rc; }
    for (int t = 0; t < n_in; t++) { pl.add_input(t); lab[t] = pl.T[t].idx; removed[t] = pl.T[t].removed; }
    for (int s = 0; s < S; s++) {
      const int Li = pl.tl[s], Ri = pl.tr[s], Oi = n_in + s;
      if ((rc = pl.do_step((size_t)s))) { err = e2; return rc; }
      cons[Li] = cons[Ri] = s;
      removed[Oi] = pl.T[Oi].removed;
      lab[Oi] = pl.T[Oi].idx;
      if (!removed[Oi] && (removed[Li] || removed[Ri])) alias[Oi] = removed[Li] ? Ri : Li;
      else if (!removed[Oi])
        for (int side = 0; side < 2; side++)
          for (int v : lab[side ? Ri : Li]) if (pos_of(lab[Oi], v) < 0) sum_step[v] = s;
    }
  }
  auto canon = [&](int t) { while (alias[t] >= 0) t = alias[t]; return t; };
  auto prod = [&](int t) { return t < n_in ? -1 : t - n_in; };
  // last consumption of a storage = consumption of the last tensor id of its alias chain
  std::vector<int> last_cons((size_t)n_t, -1), last_id((size_t)n_t, -1);
  for (int t = 0; t < n_t; t++) if (!removed[t]) { int c = canon(t); if (cons[t] >= last_cons[c]) { last_cons[c] = cons[t]; last_id[c] = t; } }

  // ---- segments: merged lifetimes of the storages above T_target
  std::vector<std::pair<int, int>> iv;
  for (int t = n_in; t < n_t; t++)
    if (!removed[t] && alias[t] < 0 && (int)lab[t].size() > cap_rank) iv.push_back({prod(t), std::min(last_cons[t], S - 1)});
  std::sort(iv.begin(), iv.end());
  struct SegSel { int a, b; std::vector<int32_t> F; int acc_id = -1; };
  std::vector<SegSel> sel;
  for (size_t i = 0; i < iv.size();) {
    int a = iv[i].first, b = iv[i].second;
    size_t j = i + 1;
    while (true) {
      while (j < iv.size() && iv[j].first <= b + 1) { b = std::max(b, iv[j].second); j++; }
      // choose F among the labels summed inside [a, b]
      std::vector<int> big;                                   // oversize storages of the segment
      for (int t = n_in + a; t <= n_in + b; t++) if (!removed[t] && alias[t] < 0 && (int)lab[t].size() > cap_rank) big.push_back(t);
      std::vector<char> inF(P.n, 0);
      std::vector<int32_t> F;
      auto need = [&]() { long r = 0; for (int t : big) { int c = 0; for (int v : lab[t]) c += inF[v]; r += std::max(0, (int)lab[t].size() - cap_rank - c); } return r; };
      long cur = need();
      bool stuck = false;
      while (cur > 0) {
        int bestv = -1; long bestgain = 0, bestocc = -1;
        std::vector<long> gain(P.n, 0), occ(P.n, 0);
        for (int t : big) {
          int c = 0; for (int v : lab[t]) c += inF[v];
          const bool over = (int)lab[t].size() - cap_rank - c > 0;
          for (int v : lab[t]) if (!inF[v] && sum_step[v] >= a && sum_step[v] <= b) { if (over) gain[v]++; occ[v]++; }
        }
        for (int v = 0; v < P.n; v++)
          if (gain[v] > bestgain || (gain[v] == bestgain && gain[v] > 0 && occ[v] > bestocc)) { bestv = v; bestgain = gain[v]; bestocc = occ[v]; }
        if (bestv < 0) { stuck = true; break; }
        inF[bestv] = 1; F.push_back(bestv);
        cur = need();
      }
      bool extend = stuck;
      int acc_id = -1;
      if (!stuck) {
        for (size_t q = 0; q < F.size();) {                   // drop indices that turned out redundant
          inF[F[q]] = 0;
          if (need() == 0) F.erase(F.begin() + (long)q); else { inF[F[q]] = 1; q++; }
        }
        // exactly one tensor that leaves the segment may depend on F
        std::vector<char> dep((size_t)n_t, 0);
        auto carries = [&](int t) { for (int v : lab[t]) if (inF[v]) return true; return false; };
        int n_out = 0;
        for (int s = a; s <= b; s++) {
          const int Li = P.tree_l[s], Ri = P.tree_r[s], Oi = n_in + s;
          for (int t : {Li, Ri}) {
            if (t < n_in) {                                   // an input consumed inside: depends on F if an endpoint is in F
              const int u = t < P.m ? P.eu[t] : t - P.m, v = t < P.m ? P.ev[t] : -1;
              if (inF[u] || (v >= 0 && inF[v])) dep[t] = 1;
            } else if (prod(t) < a && !removed[t] && carries(t)) dep[t] = 1;
          }
          dep[Oi] = dep[Li] || dep[Ri];
        }
        for (int t = n_in + a; t <= n_in + b; t++)
          if (dep[t] && !removed[t] && cons[t] > b) { n_out++; acc_id = t; }
        if (n_out != 1) extend = true;
      }
      if (!extend) {
        if (F.size() > 24) { err = "a segment needs more than 24 locally fixed indices"; return ST_ESHAPE; }
        sel.push_back({a, b, F, acc_id});
        break;
      }
      if (b >= S - 1) { err = "the tree joins two sliced parts: no local fixed set brings the segment under T_target"; return ST_ESHAPE; }
      b++;
    }
    i = j;
  }

  // ---- pass 1: the walk that emits steps and assigns storage
  // two arenas: tensors that depend on a stretch's fixed indices are leaf-variant (one copy per branch of the batch
  // in flight), everything else -- in particular every tensor that crosses a stretch boundary -- is invariant
  Planner pl(P, 1, false, false, false, out.plan, err);
  int rc;
  pl.cap_rank = cap_rank;
  pl.set_fixed({}); pl.count_occurrences();
  if ((rc = pl.init_tree({}))) return rc;
  std::vector<std::vector<int>> inputs_of((size_t)S);        // inputs by the step that consumes them
  for (int t = 0; t < n_in; t++) if (cons[t] < S) inputs_of[cons[t]].push_back(t);
  auto run_range = [&](int a, int b, LocalSeg &ls) -> int {
    ls.step_begin = (int32_t)out.plan.steps.size();
    for (int s = a; s <= b; s++)
      for (int t : inputs_of[s]) {
        pl.add_input(t);
        const InputRec &r = out.plan.inputs[t];
        (r.rank == 0 ? ls.list_scalar : (r.variant ? ls.list_var : ls.list_inv)).push_back(t);
      }
    if (n_in == 1 && a == 0) { pl.add_input(0); (out.plan.inputs[0].rank == 0 ? ls.list_scalar : ls.list_inv).push_back(0); }
    for (int s = a; s <= b; s++) if ((rc = pl.do_step((size_t)s))) return rc;
    ls.step_end = (int32_t)out.plan.steps.size();
    for (int q = ls.step_begin; q < ls.step_end; q++) {
      const Step &st = out.plan.steps[q];
      ls.fma += st.fma; ls.bytes += st.bytes;
      ls.max_rank = std::max(ls.max_rank, std::max(st.rO, std::max(st.rA, st.rB)));
    }
    return 0;
  };
  int next = 0;
  for (size_t q = 0; q <= sel.size(); q++) {
    const int a = q < sel.size() ? sel[q].a : S, b = q < sel.size() ? sel[q].b : S - 1;
    if (next < a || (S == 0 && q == 0)) {                     // the stretch before the segment: runs once
      LocalSeg ls;
      if ((rc = run_range(next, a - 1, ls))) return rc;
      out.segs.push_back(std::move(ls));
    }
    if (q == sel.size()) break;
    LocalSeg ls;
    ls.fixed = sel[q].F;
    std::vector<char> inF(P.n, 0);
    for (int v : ls.fixed) inF[v] = 1;
    // tensors that enter the segment stay in storage until its last slice; those carrying F become views
    std::vector<std::pair<int64_t, int64_t>> bases;
    for (int t = n_in; t < n_in + a; t++) {                   // produced before the segment (inputs are built by the segment that consumes them)
      TRef &x = pl.T[t];
      if (pl.used[t] || x.removed) continue;
      if (cons[t] > b) continue;                              // passes the segment untouched
      bool hit = false;
      for (int v : x.idx) if (inF[v]) hit = true;
      if (x.variant) { err = "internal: a branch-dependent tensor crosses a stretch boundary"; return ST_EINVAL; }
      if (!hit) { x.keep = true; continue; }
      bases.push_back({x.off, (int64_t)1 << x.idx.size()});
      TRef vw = x;
      vw.idx.clear(); vw.phys.clear(); vw.slice.assign(ls.fixed.size(), 0u);
      for (size_t p2 = 0; p2 < x.idx.size(); p2++) {
        const int v = x.idx[p2];
        if (inF[v]) { vw.slice[(size_t)pos_of(ls.fixed, v)] = Planner::bit_of(x, (int)p2); vw.sub.erase(v); }
        else { vw.idx.push_back(v); vw.phys.push_back(Planner::bit_of(x, (int)p2)); }
      }
      vw.ext = true; vw.keep = false; vw.variant = true;     // read per branch: its consumers are branch-dependent
      x = std::move(vw);
    }
    const int acc_id = sel[q].acc_id;
    ls.acc_rank = (int32_t)lab[acc_id].size();
    ls.acc_off = pl.ai.alloc((int64_t)1 << ls.acc_rank);
    std::vector<int32_t> F32(ls.fixed.begin(), ls.fixed.end());
    if ((rc = pl.set_fixed(F32))) return rc;
    pl.deferred.clear();
    if ((rc = run_range(a, b, ls))) return rc;
    pl.set_fixed({});
    // the per-slice result sits at tmp_off; the tensor the rest of the tree sees is the accumulator
    TRef &z = pl.T[acc_id];
    if (z.removed || (int)z.idx.size() != ls.acc_rank || z.ext || !z.variant) { err = "internal: sliced segment lost its result tensor"; return ST_EINVAL; }
    for (int v : z.idx) if (inF[v]) { err = "internal: a locally fixed index leaves its segment"; return ST_EINVAL; }
    ls.tmp_off = z.off;
    pl.av.release(z.off, (int64_t)1 << ls.acc_rank);
    z.off = ls.acc_off; z.variant = false;                    // (+) over the branches: no longer branch-dependent
    for (auto &bo : bases) pl.ai.release(bo.first, bo.second);
    for (auto &d : pl.deferred) (d.variant ? pl.av : pl.ai).release(d.off, d.ne);
    pl.deferred.clear();
    for (int t = 0; t <= n_in + b; t++) {
      TRef &x = pl.T[t];
      if (pl.used[t] || x.removed) continue;
      x.keep = false;
      if (x.variant) { err = "internal: a branch-dependent tensor is still live after its segment"; return ST_EINVAL; }
      for (int v : x.idx) if (inF[v]) { err = "internal: a locally fixed index is still open after its segment"; return ST_EINVAL; }
    }
    ls.bytes += 36.0 * (double)((int64_t)1 << ls.acc_rank);   // accumulation pass: read slice + read/write accumulator
    out.max_fixed = std::max<int32_t>(out.max_fixed, (int32_t)ls.fixed.size());
    out.n_sliced_segs++;
    out.segs.push_back(std::move(ls));
    next = b + 1;
  }
  for (const LocalSeg &ls : out.segs) {
    const double ns = std::ldexp(1.0, (int)ls.fixed.size());
    out.fma_total += ns * ls.fma; out.bytes_total += ns * ls.bytes; out.n_slices += ns;
  }
  return pl.finish();
}

}  // namespace bbtn
