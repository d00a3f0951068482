// bound_api.cu -- bbtn_region_bound (tables for K5) and bbtn_solve_bb (host branch/prune loop, S6).
// Host logic only: bounds come from K5 (bound.cu), leaf values from K1..K4.
#include <algorithm>
#include <cstring>
#include <numeric>

#include "handle.h"

using namespace bbtn;

namespace {

int build_bound_plan(bbtn_handle *h, const int32_t *roff, const int32_t *rv, int n_regions,
                     const int32_t *fixed, int n_fixed, BoundPlan **out) {
  std::vector<int32_t> key;
  key.push_back(n_regions);
  if (n_regions > 0) { key.insert(key.end(), roff, roff + n_regions + 1); key.insert(key.end(), rv, rv + roff[n_regions]); }
  key.push_back(-1);
  key.insert(key.end(), fixed, fixed + n_fixed);
  auto it = h->bounds.find(key);
  if (it != h->bounds.end()) { *out = it->second.get(); return BBTN_OK; }

  const Problem &P = h->P;
  std::vector<int> fpos(P.n, -1), reg(P.n, -1), lb(P.n, -1);
  for (int j = 0; j < n_fixed; j++) {
    if (fixed[j] < 0 || fixed[j] >= P.n) return fail(h, BBTN_EINVAL, "fixed vertex id out of range");
    if (fpos[fixed[j]] >= 0) return fail(h, BBTN_EINVAL, "duplicate fixed vertex");
    fpos[fixed[j]] = j;
  }
  std::vector<int32_t> reg_off(1, 0), reg_vw;
  for (int j = 0; j < n_regions; j++) {
    if (roff[j + 1] < roff[j]) return fail(h, BBTN_EINVAL, "region_offsets must be non-decreasing");
    int nf = 0;
    for (int p = roff[j]; p < roff[j + 1]; p++) {
      int v = rv[p];
      if (v < 0 || v >= P.n) return fail(h, BBTN_EINVAL, "region vertex id out of range");
      if (fpos[v] >= 0) continue;
      if (reg[v] >= 0) return fail(h, BBTN_EINVAL, "regions must be disjoint");
      reg[v] = j; lb[v] = nf++; reg_vw.push_back(P.vw[v]);
    }
    if (nf > 20) return fail(h, BBTN_EINVAL, "a region may hold at most 20 free vertices");
    reg_off.push_back((int32_t)reg_vw.size());
  }
  std::vector<std::vector<int32_t>> fx_bit(n_regions), fx_col(n_regions), fx_w(n_regions), pr_a(n_regions), pr_b(n_regions), pr_w(n_regions);
  std::vector<int32_t> ff_cu, ff_cv, ff_w, fv_c, fv_w;
  std::vector<std::vector<int32_t>> nbr_cols(P.n);
  int64_t cst = 0;
  const bool ising = P.kind == 0;
  for (int e = 0; e < P.m; e++) {
    const int u = P.eu[e], v = P.ev[e], w = P.ew[e];
    const bool fu = fpos[u] >= 0, fv = fpos[v] >= 0;
    if (fu && fv) { ff_cu.push_back(fpos[u]); ff_cv.push_back(fpos[v]); ff_w.push_back(w); continue; }
    if (fu != fv) {
      const int fr = fu ? v : u, fxd = fu ? u : v;
      if (reg[fr] >= 0) { fx_bit[reg[fr]].push_back(lb[fr]); fx_col[reg[fr]].push_back(fpos[fxd]); fx_w[reg[fr]].push_back(w); }
      else { if (ising) cst += std::abs(w); else nbr_cols[fr].push_back(fpos[fxd]); }
      continue;
    }
    if (reg[u] >= 0 && reg[u] == reg[v]) { pr_a[reg[u]].push_back(lb[u]); pr_b[reg[u]].push_back(lb[v]); pr_w[reg[u]].push_back(w); }
    else if (ising) cst += std::abs(w);
  }
  std::vector<int32_t> uv_off(1, 0), uv_cols, uv_w;
  for (int i = 0; i < P.n; i++) {
    if (fpos[i] >= 0) { fv_c.push_back(fpos[i]); fv_w.push_back(P.vw[i]); continue; }
    if (reg[i] >= 0) continue;
    if (ising) cst += std::abs(P.vw[i]);
    else if (nbr_cols[i].empty()) cst += std::max(P.vw[i], 0);
    else { uv_cols.insert(uv_cols.end(), nbr_cols[i].begin(), nbr_cols[i].end()); uv_off.push_back((int32_t)uv_cols.size()); uv_w.push_back(P.vw[i]); }
  }
  if (cst > BBTN_ENERGY_LIMIT) return fail(h, BBTN_ERANGE, "bound constant out of range");
  auto flat = [&](const std::vector<std::vector<int32_t>> &vv, std::vector<int32_t> &o, std::vector<int32_t> *off) {
    if (off) off->assign(1, 0);
    for (auto &v : vv) { o.insert(o.end(), v.begin(), v.end()); if (off) off->push_back((int32_t)o.size()); }
  };
  std::vector<int32_t> fxo, fxb, fxc, fxw, pro, pa, pb, pw;
  flat(fx_bit, fxb, &fxo); flat(fx_col, fxc, nullptr); flat(fx_w, fxw, nullptr);
  flat(pr_a, pa, &pro); flat(pr_b, pb, nullptr); flat(pr_w, pw, nullptr);

  auto bp = std::make_unique<BoundPlan>();
  BoundTables &t = bp->t;
  std::memset(&t, 0, sizeof(t));
  t.kind = P.kind; t.n_regions = n_regions; t.n_fixed = n_fixed; t.const_term = (int32_t)cst;
  int k = 0;
  auto up = [&](const std::vector<int32_t> &v, const int32_t *&dst) -> cudaError_t {
    cudaError_t e = bp->tab[k].upload(v);
    dst = (const int32_t *)bp->tab[k].p; k++;
    return e;
  };
  CUDA_TRY(h, up(reg_off, t.reg_off)); CUDA_TRY(h, up(reg_vw, t.reg_vw));
  CUDA_TRY(h, up(fxo, t.reg_fix_off)); CUDA_TRY(h, up(fxb, t.reg_fix_bit)); CUDA_TRY(h, up(fxc, t.reg_fix_col)); CUDA_TRY(h, up(fxw, t.reg_fix_w));
  CUDA_TRY(h, up(pro, t.reg_pair_off)); CUDA_TRY(h, up(pa, t.reg_pair_a)); CUDA_TRY(h, up(pb, t.reg_pair_b)); CUDA_TRY(h, up(pw, t.reg_pair_w));
  t.n_ff = (int)ff_w.size(); CUDA_TRY(h, up(ff_cu, t.ff_cu)); CUDA_TRY(h, up(ff_cv, t.ff_cv)); CUDA_TRY(h, up(ff_w, t.ff_w));
  t.n_fv = (int)fv_w.size(); CUDA_TRY(h, up(fv_c, t.fv_c)); CUDA_TRY(h, up(fv_w, t.fv_w));
  t.n_uf = 0;
  t.n_uv = (int)uv_w.size(); CUDA_TRY(h, up(uv_off, t.uv_off)); CUDA_TRY(h, up(uv_cols, t.uv_cols)); CUDA_TRY(h, up(uv_w, t.uv_w));
  if (h->bounds.size() > 64) h->bounds.clear();          // B&B levels come and go; keep the cache small
  *out = bp.get();
  h->bounds.emplace(key, std::move(bp));
  return BBTN_OK;
}

}  // namespace

extern "C" {

int bbtn_oplus_combine(int32_t kind, int64_t n, const int32_t *energy, const uint64_t *count, const uint32_t *count_mod,
                       int32_t *out_energy, uint64_t *out_count, uint32_t *out_count_mod);
}

namespace {
struct BB {
  bbtn_handle *h; cudaStream_t st;
  const int32_t *branch; int n_branch, chunk;
  const int32_t *roff, *rv; int n_regions;
  int64_t max_batch; bool prune; bool ising, crt;
  bool have_inc = false; int32_t inc = 0;         // best energy known (hint or found), reported units
  bool have_best = false; int32_t best = 0; uint64_t cnt = 0; uint64_t m1 = 0, m2 = 0;
  int64_t stats[4] = {0, 0, 0, 0};

  bool worse(int32_t bound) const { return ising ? bound > inc : bound < inc; }   // strictly (reading A14)

  int contract(const std::vector<uint8_t> &asg, int64_t B, int d) {
    std::vector<int32_t> e((size_t)B); std::vector<uint64_t> c((size_t)B); std::vector<uint32_t> cm(crt ? (size_t)B * 2 : 0);
    int rc = bbtn_contract_batch(h, branch, d, asg.data(), B, e.data(), c.data(), crt ? cm.data() : nullptr, st);
    if (rc) return rc;
    stats[2] += B; stats[3] += 1;
    // (+) over the batch, then into the running result (Eq. 3's outer sum)
    int32_t e2[2] = {have_best ? best : BBTN_NEG_INF, BBTN_NEG_INF}; uint64_t c2[2] = {cnt, 0}; uint32_t cm2[4] = {(uint32_t)m1, (uint32_t)m2, 0, 0};
    rc = bbtn_oplus_combine(ising ? BBTN_ISING : BBTN_MIS, B, e.data(), c.data(), crt ? cm.data() : nullptr, &e2[1], &c2[1], crt ? &cm2[2] : nullptr);
    if (rc) return rc;
    uint32_t om[2] = {0, 0};
    rc = bbtn_oplus_combine(ising ? BBTN_ISING : BBTN_MIS, 2, e2, c2, crt ? cm2 : nullptr, &best, &cnt, crt ? om : nullptr);
    if (rc) return rc;
    m1 = om[0]; m2 = om[1];
    have_best = best != BBTN_NEG_INF;
    if (have_best && (!have_inc || (ising ? best < inc : best > inc))) { inc = best; have_inc = true; }
    return BBTN_OK;
  }

  // parents: [np][d] assignments of the first d branch vertices
  int expand(const std::vector<uint8_t> &parents, int64_t np, int d) {
    const int d2 = std::min(d + chunk, n_branch), c = d2 - d;
    const int64_t nc = np << c;
    std::vector<uint8_t> kids((size_t)nc * d2);
    for (int64_t p = 0; p < np; p++)
      for (int64_t x = 0; x < ((int64_t)1 << c); x++) {
        uint8_t *row = &kids[(size_t)((p << c) + x) * d2];
        if (d) std::memcpy(row, &parents[(size_t)p * d], (size_t)d);
        for (int j = 0; j < c; j++) row[d + j] = (uint8_t)((x >> j) & 1);
      }
    stats[0] += nc;
    std::vector<int32_t> bound((size_t)nc);
    int rc = bbtn_region_bound(h, roff, rv, n_regions, branch, d2, kids.data(), nc, bound.data(), st);
    if (rc) return rc;
    std::vector<int64_t> keep;
    for (int64_t i = 0; i < nc; i++) {
      if (bound[i] == BBTN_NEG_INF && !ising) { stats[1]++; continue; }          // infeasible
      if (prune && have_inc && worse(bound[i])) { stats[1]++; continue; }
      keep.push_back(i);
    }
    std::stable_sort(keep.begin(), keep.end(), [&](int64_t a, int64_t b) { return ising ? bound[a] < bound[b] : bound[a] > bound[b]; });
    const bool last = d2 == n_branch;
    const int64_t slice = last ? max_batch : std::max<int64_t>(1, max_batch >> std::min(chunk, 20));
    for (size_t s0 = 0; s0 < keep.size();) {
      std::vector<uint8_t> sub; int64_t ns = 0;
      while (s0 < keep.size() && ns < slice) {
        const int64_t i = keep[s0++];
        if (prune && have_inc && worse(bound[i])) { stats[1]++; continue; }      // incumbent may have improved
        sub.insert(sub.end(), &kids[(size_t)i * d2], &kids[(size_t)i * d2] + d2); ns++;
      }
      if (ns == 0) continue;
      rc = last ? contract(sub, ns, d2) : expand(sub, ns, d2);
      if (rc) return rc;
    }
    return BBTN_OK;
  }
};
}  // namespace

extern "C" {

int bbtn_region_bound(bbtn_handle *h, const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions,
                      const int32_t *fixed, int32_t n_fixed, const uint8_t *assign, int64_t B, int32_t *bound, void *stream) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  if (B < 1 || !bound || n_regions < 0 || n_fixed < 0 || (n_regions > 0 && (!region_offsets || !region_vertices)) ||
      (n_fixed > 0 && (!fixed || !assign)))
    return fail(h, BBTN_EINVAL, "bad region_bound arguments");
  if (!have_device()) return fail(h, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  BoundPlan *bp = nullptr;
  int rc = build_bound_plan(h, region_offsets, region_vertices, n_regions, fixed, n_fixed, &bp);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const bool dev_io = (h->P.flags & BBTN_IO_DEVICE) != 0;
  CUDA_TRY(h, bp->scratch.ensure((size_t)B * std::max(n_regions, 1) * 4));
  const uint8_t *d_assign = assign; int32_t *d_bound = bound;
  if (!dev_io) {
    CUDA_TRY(h, bp->assign.ensure((size_t)B * std::max(n_fixed, 1)));
    CUDA_TRY(h, bp->bound.ensure((size_t)B * 4));
    if (n_fixed > 0) CUDA_TRY(h, cudaMemcpyAsync(bp->assign.p, assign, (size_t)B * n_fixed, cudaMemcpyHostToDevice, st));
    d_assign = (const uint8_t *)bp->assign.p; d_bound = (int32_t *)bp->bound.p;
  }
  launch_region_bound(bp->t, d_assign, B, (int32_t *)bp->scratch.p, d_bound, st);
  CUDA_TRY(h, cudaGetLastError());
  if (!dev_io) {
    std::vector<int32_t> tmp((size_t)B);
    CUDA_TRY(h, cudaMemcpyAsync(tmp.data(), d_bound, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(h, cudaStreamSynchronize(st));
    std::memcpy(bound, tmp.data(), (size_t)B * 4);
  }
  return BBTN_OK;
}

int bbtn_region_bound_static(bbtn_handle *h, const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions,
                             const int32_t *fixed, int32_t n_fixed, const uint8_t *assign, int64_t B, int32_t *bound, void *stream) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  if (B < 0 || (B > 0 && !bound) || n_regions < 0 || n_fixed < 0 || (n_regions > 0 && (!region_offsets || !region_vertices)) ||
      (n_fixed > 0 && (!fixed || (B > 0 && !assign))))
    return fail(h, BBTN_EINVAL, "bad region_bound_static arguments");
  if ((double)B * (double)std::max(n_regions, 1) > (double)BBTN_REGION_BOUND_STATIC_MAX_ITEMS)
    return fail(h, BBTN_ESHAPE, "bbtn_region_bound_static: B * n_regions = " + std::to_string(B) + " * " + std::to_string(std::max(n_regions, 1)) +
                                    " exceeds the static scratch of " + std::to_string(BBTN_REGION_BOUND_STATIC_MAX_ITEMS) +
                                    " entries; split the batch or use bbtn_region_bound");
  if (!have_device()) return fail(h, BBTN_ECUDA, "no CUDA device (there is no CPU fallback)");
  // look the tables up, never build them (building uploads = allocates)
  std::vector<int32_t> key;
  key.push_back(n_regions);
  if (n_regions > 0) { key.insert(key.end(), region_offsets, region_offsets + n_regions + 1); key.insert(key.end(), region_vertices, region_vertices + region_offsets[n_regions]); }
  key.push_back(-1);
  key.insert(key.end(), fixed, fixed + n_fixed);
  auto it = h->bounds.find(key);
  if (it == h->bounds.end())
    return fail(h, BBTN_EINVAL, "bbtn_region_bound_static: no cached tables for these regions and fixed vertices; call bbtn_region_bound with them once first");
  cudaError_t ce = cudaSuccess;
  // B = 0: set-up only (the launcher resolves the array's address for this device and launches nothing)
  const int rc = launch_region_bound_static(it->second->t, assign, B, bound, (cudaStream_t)stream, &ce);
  if (rc == 2) return fail(h, BBTN_ECUDA, "bbtn_region_bound_static: device ordinal beyond 63");
  if (rc) return fail(h, BBTN_ECUDA, std::string("bbtn_region_bound_static: ") + cudaGetErrorString(ce));
  CUDA_TRY(h, cudaGetLastError());
  return BBTN_OK;
}

int bbtn_oplus_combine(int32_t kind, int64_t n, const int32_t *energy, const uint64_t *count, const uint32_t *count_mod,
                       int32_t *out_energy, uint64_t *out_count, uint32_t *out_count_mod) {
  if ((kind != BBTN_ISING && kind != BBTN_MIS) || n < 0 || (n > 0 && (!energy || !count)) || !out_energy || !out_count ||
      (out_count_mod && n > 0 && !count_mod))
    return fail(nullptr, BBTN_EINVAL, "bad oplus_combine arguments");
  bool have = false; int32_t best = BBTN_NEG_INF; uint64_t cnt = 0, m1 = 0, m2 = 0;
  for (int64_t b = 0; b < n; b++) {
    if (energy[b] == BBTN_NEG_INF) continue;
    if (!have || (kind == BBTN_ISING ? energy[b] < best : energy[b] > best)) { best = energy[b]; cnt = 0; m1 = m2 = 0; have = true; }
    if (energy[b] == best) {
      cnt += count[b];
      if (out_count_mod) { m1 = (m1 + count_mod[2 * b]) % BBTN_P1; m2 = (m2 + count_mod[2 * b + 1]) % BBTN_P2; }
    }
  }
  *out_energy = have ? best : BBTN_NEG_INF;
  *out_count = have ? cnt : 0;
  if (out_count_mod) { out_count_mod[0] = (uint32_t)m1; out_count_mod[1] = (uint32_t)m2; }
  return BBTN_OK;
}

int bbtn_solve_bb(bbtn_handle *h, const int32_t *branch_vertices, int32_t n_branch, int32_t chunk,
                  const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions,
                  int64_t max_batch, int32_t incumbent_hint, int32_t use_pruning,
                  int32_t *energy, uint64_t *count, uint32_t *count_mod, int64_t *stats, void *stream) {
  if (!h) return fail(nullptr, BBTN_EINVAL, "null handle");
  if (n_branch < 0 || (n_branch > 0 && !branch_vertices) || chunk < 1 || chunk > 20 || max_batch < 1 || !energy || !count)
    return fail(h, BBTN_EINVAL, "bad solve_bb arguments");
  if (h->P.flags & BBTN_IO_DEVICE) return fail(h, BBTN_EINVAL, "bbtn_solve_bb needs a host-pointer handle");
  const bool crt = (h->P.flags & BBTN_COUNT_CRT) != 0;
  if (count_mod && !crt) return fail(h, BBTN_EINVAL, "count_mod needs a handle built with BBTN_COUNT_CRT");
  BB bb{h, (cudaStream_t)stream, branch_vertices, n_branch, chunk, region_offsets, region_vertices, n_regions,
        max_batch, use_pruning != 0, h->P.kind == BBTN_ISING, crt && count_mod != nullptr};
  if (incumbent_hint != BBTN_NEG_INF) { bb.have_inc = true; bb.inc = incumbent_hint; }
  int rc;
  if (n_branch == 0) {
    std::vector<uint8_t> none;
    bb.stats[0] = 1;
    rc = bb.contract(none, 1, 0);
  } else {
    std::vector<uint8_t> root;
    rc = bb.expand(root, 1, 0);
  }
  if (rc) return rc;
  *energy = bb.have_best ? bb.best : BBTN_NEG_INF;
  *count = bb.have_best ? bb.cnt : 0;
  if (count_mod) { count_mod[0] = (uint32_t)bb.m1; count_mod[1] = (uint32_t)bb.m2; }
  if (stats) std::memcpy(stats, bb.stats, sizeof(bb.stats));
  return BBTN_OK;
}

}  // extern "C"
