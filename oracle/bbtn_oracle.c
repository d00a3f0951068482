/*
 * bbtn_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU restatement of what the BBTN hot path
 * computes (arxiv/paper_2602_05470).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may call it.  It shares no
 * code, header, table or constant with paper_2602_05470_b200/csrc.
 *
 * Representation is deliberately unlike the GPU's: energies are int64, the
 * semiring zero ("the tuple (inf, 0)") is an explicit flag, and
 * counts are 256-bit unsigned integers (four 64-bit limbs, little endian), so
 * no sentinel trick and no wrap-around can hide a mistake.
 *
 * Everything is max-plus on negated Ising energies (reading A1): the
 * paper writes min-sum ("x (+) y = min(x,y), x (.) y = x+y"); the two
 * are mirror images.  Functions:
 *
 *   oracle_exhaustive      Eq. 1 / Eq. 2 evaluated literally: loop over every
 *                          configuration (MIS PAPER.md:55).
 *   oracle_contract_tree   Eq. 2 evaluated pairwise along an SSA tree with naive
 *                          loop nests, sliced per Eq. 3 (:61).
 *   oracle_frontier_dp     independent exact method: vertex-by-vertex transfer
 *                          (frontier) dynamic programme in the same algebra.
 *   oracle_frontier_dp_mis_sparse  the same programme for MIS with only the
 *                          independent frontier states stored (large King's subgraphs).
 *   oracle_gemm            C[b,m,n] = (+)_k A[b,m,k] (.) B[b,k,n], triple loop.
 *   oracle_permute         dst[pi(i)] = src[i] for a bit permutation pi.
 *   oracle_region_bound    DESIGN.md reading A15 of the pruning bound
 *                          (PAPER.md:65-67), written out literally.
 *   oracle_rho             Eq. 4 for a list of tensor ranks.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms, brute force,
 * invariants, library routines; see DESIGN.md "Oracle pins".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint64_t w[4]; } u256;

static u256 u256_from(uint64_t x) { u256 r = {{x, 0, 0, 0}}; return r; }
static u256 u256_add(u256 a, u256 b) {
    u256 r; unsigned __int128 c = 0;
    for (int i = 0; i < 4; i++) { c += (unsigned __int128)a.w[i] + b.w[i]; r.w[i] = (uint64_t)c; c >>= 64; }
    return r;
}
static u256 u256_mul(u256 a, u256 b) {            /* product mod 2^256 */
    u256 r = {{0, 0, 0, 0}};
    for (int i = 0; i < 4; i++) {
        unsigned __int128 c = 0;
        for (int j = 0; i + j < 4; j++) {
            c += (unsigned __int128)a.w[i] * b.w[j] + r.w[i + j];
            r.w[i + j] = (uint64_t)c; c >>= 64;
        }
    }
    return r;
}

/* one semiring element */
typedef struct { int64_t e; int zero; u256 c; } elem;
static elem el_zero(void) { elem r; r.e = 0; r.zero = 1; r.c = u256_from(0); return r; }
static elem el_make(int64_t e, uint64_t c) { elem r; r.e = e; r.zero = 0; r.c = u256_from(c); return r; }
/* (a,ca) (.) (b,cb) = (a+b, ca*cb); zero absorbs */
static elem el_mul(elem a, elem b) {
    if (a.zero || b.zero) return el_zero();
    elem r; r.e = a.e + b.e; r.zero = 0; r.c = u256_mul(a.c, b.c); return r;
}
/* (a,ca) (+) (b,cb): larger energy wins, counts add on ties; zero is neutral */
static elem el_add(elem a, elem b) {
    if (a.zero) return b;
    if (b.zero) return a;
    if (a.e > b.e) return a;
    if (b.e > a.e) return b;
    elem r; r.e = a.e; r.zero = 0; r.c = u256_add(a.c, b.c); return r;
}

/* ---- input tensors (PAPER.md:49 Ising, :55 MWIS), max-plus form ------------
 * Ising: s=0 <-> sigma=-1, s=1 <-> sigma=+1 (reading A2); bond entry +J*sigma_u*sigma_v,
 *        vertex entry +h*sigma; counts 1.
 * MIS:   bond entry (0,1) except [1][1] = zero element; vertex entry (0,1),(w,1). */
static int64_t sgn(int s) { return 2 * s - 1; }
static elem bond_entry(int kind, int64_t J, int su, int sv) {
    if (kind == 0) return el_make(J * sgn(su) * sgn(sv), 1);
    return (su == 1 && sv == 1) ? el_zero() : el_make(0, 1);
}
static elem vertex_entry(int kind, int64_t w, int s) {
    if (kind == 0) return el_make(w * sgn(s), 1);
    return el_make(s ? w : 0, 1);
}
static int64_t ew_of(const int32_t *edge_w, int e) { return edge_w ? edge_w[e] : 1; }
static int64_t vw_of(int kind, const int32_t *vertex_w, int i) {
    if (vertex_w) return vertex_w[i];
    return kind == 0 ? 0 : 1;          /* no field / unit weight */
}

static void write_out(elem r, int kind, int64_t *energy, int32_t *feasible, uint64_t *count4) {
    *feasible = !r.zero;
    /* Ising: reported energy is min H = -(max-plus value); MIS: the weight itself */
    *energy = r.zero ? 0 : (kind == 0 ? -r.e : r.e);
    for (int i = 0; i < 4; i++) count4[i] = r.zero ? 0 : r.c.w[i];
}

/* ---- oracle-1: the definition ------------------------------------------------ */
int oracle_exhaustive(int kind, int n, int m, const int32_t *eu, const int32_t *ev,
                      const int32_t *edge_w, const int32_t *vertex_w,
                      int n_fixed, const int32_t *fixed, const uint8_t *assign,
                      int64_t *energy, int32_t *feasible, uint64_t *count4)
{
    if (n - n_fixed > 30) return 1;
    int *val = (int *)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
    int *freev = (int *)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
    for (int i = 0; i < n; i++) val[i] = -1;
    for (int j = 0; j < n_fixed; j++) val[fixed[j]] = assign[j] ? 1 : 0;
    int nf = 0;
    for (int i = 0; i < n; i++) if (val[i] < 0) freev[nf++] = i;
    elem best = el_zero();
    for (uint64_t x = 0; x < (1ull << nf); x++) {
        for (int j = 0; j < nf; j++) val[freev[j]] = (int)((x >> j) & 1);
        int64_t tot = 0; int ok = 1;
        if (kind == 0) {
            /* Eq. 1 with the sign flipped: -H(sigma) = sum J s s + sum h s */
            for (int e = 0; e < m; e++) tot += ew_of(edge_w, e) * sgn(val[eu[e]]) * sgn(val[ev[e]]);
            for (int i = 0; i < n; i++) tot += vw_of(kind, vertex_w, i) * sgn(val[i]);
        } else {
            for (int e = 0; e < m && ok; e++) if (val[eu[e]] && val[ev[e]]) ok = 0;
            for (int i = 0; i < n; i++) if (val[i]) tot += vw_of(kind, vertex_w, i);
        }
        if (ok) best = el_add(best, el_make(tot, 1));
    }
    write_out(best, kind, energy, feasible, count4);
    free(val); free(freev);
    return 0;
}

/* ---- oracle-2: naive loop-nest contraction along the given tree -------------- */
typedef struct { int rank; int *idx; elem *v; } tensor;   /* idx[p] <-> bit p of the linear index */

static void tensor_free(tensor *t) { free(t->idx); free(t->v); t->idx = NULL; t->v = NULL; }

int oracle_contract_tree(int kind, int n, int m, const int32_t *eu, const int32_t *ev,
                         const int32_t *edge_w, const int32_t *vertex_w,
                         int n_steps, const int32_t *tree_l, const int32_t *tree_r,
                         int n_fixed, const int32_t *fixed, const uint8_t *assign,
                         int64_t *energy, int32_t *feasible, uint64_t *count4, int32_t *max_rank)
{
    int n_in = m + n;
    if (n_steps != n_in - 1) return 2;
    int *val = (int *)malloc(sizeof(int) * (size_t)(n + 1));
    for (int i = 0; i < n; i++) val[i] = -1;
    for (int j = 0; j < n_fixed; j++) val[fixed[j]] = assign[j] ? 1 : 0;
    int total = n_in + n_steps;
    tensor *T = (tensor *)calloc((size_t)total, sizeof(tensor));
    int *occ_total = (int *)calloc((size_t)(n + 1), sizeof(int));
    /* per node: how many INPUT tensors inside its subtree carry index i -> sparse lists */
    int **sub_idx = (int **)calloc((size_t)total, sizeof(int *));
    int **sub_cnt = (int **)calloc((size_t)total, sizeof(int *));
    int *sub_n = (int *)calloc((size_t)total, sizeof(int));
    int rc = 0; *max_rank = 0;

    /* step 1+2: inputs in ABI order, sliced */
    for (int t = 0; t < n_in; t++) {
        int a[2], na = 0;
        if (t < m) { if (val[eu[t]] < 0) a[na++] = eu[t]; if (val[ev[t]] < 0) a[na++] = ev[t]; }
        else if (val[t - m] < 0) a[na++] = t - m;
        T[t].rank = na; T[t].idx = (int *)malloc(sizeof(int) * 2); T[t].v = (elem *)malloc(sizeof(elem) * 4);
        for (int p = 0; p < na; p++) { T[t].idx[p] = a[p]; occ_total[a[p]]++; }
        for (int x = 0; x < (1 << na); x++) {
            if (t < m) {
                int su = val[eu[t]], sv = val[ev[t]], p = 0;
                if (su < 0) su = (x >> p++) & 1;
                if (sv < 0) sv = (x >> p++) & 1;
                T[t].v[x] = bond_entry(kind, ew_of(edge_w, t), su, sv);
            } else {
                int s = val[t - m]; if (s < 0) s = x & 1;
                T[t].v[x] = vertex_entry(kind, vw_of(kind, vertex_w, t - m), s);
            }
        }
        sub_n[t] = na; sub_idx[t] = (int *)malloc(sizeof(int) * 2); sub_cnt[t] = (int *)malloc(sizeof(int) * 2);
        for (int p = 0; p < na; p++) { sub_idx[t][p] = a[p]; sub_cnt[t][p] = 1; }
    }
    /* step 3: SSA steps */
    for (int s = 0; s < n_steps && !rc; s++) {
        int L = tree_l[s], R = tree_r[s], O = n_in + s;
        if (L < 0 || R < 0 || L >= O || R >= O || L == R || !T[L].v || !T[R].v) { rc = 3; break; }
        /* merged subtree occurrence counts */
        int cap = sub_n[L] + sub_n[R];
        sub_idx[O] = (int *)malloc(sizeof(int) * (size_t)(cap + 1)); sub_cnt[O] = (int *)malloc(sizeof(int) * (size_t)(cap + 1));
        int k = 0;
        for (int p = 0; p < sub_n[L]; p++) { sub_idx[O][k] = sub_idx[L][p]; sub_cnt[O][k] = sub_cnt[L][p]; k++; }
        for (int p = 0; p < sub_n[R]; p++) {
            int q; for (q = 0; q < sub_n[L]; q++) if (sub_idx[O][q] == sub_idx[R][p]) break;
            if (q < sub_n[L]) sub_cnt[O][q] += sub_cnt[R][p];
            else { sub_idx[O][k] = sub_idx[R][p]; sub_cnt[O][k] = sub_cnt[R][p]; k++; }
        }
        /* I_O: indices still carried by an input tensor outside this subtree; drop finished ones */
        int kk = 0;
        for (int p = 0; p < k; p++) if (sub_cnt[O][p] < occ_total[sub_idx[O][p]]) {
            sub_idx[O][kk] = sub_idx[O][p]; sub_cnt[O][kk] = sub_cnt[O][p]; kk++; }
        sub_n[O] = kk;
        /* union of I_L and I_R */
        int un[64], nu = 0;
        for (int p = 0; p < T[L].rank; p++) un[nu++] = T[L].idx[p];
        for (int p = 0; p < T[R].rank; p++) {
            int q; for (q = 0; q < nu; q++) if (un[q] == T[R].idx[p]) break;
            if (q == nu) { if (nu >= 40) { rc = 4; break; } un[nu++] = T[R].idx[p]; }
        }
        if (rc) break;
        if (nu > 34) { rc = 4; break; }
        /* output indices = union members that are in I_O */
        T[O].idx = (int *)malloc(sizeof(int) * (size_t)(nu + 1)); T[O].rank = 0;
        for (int q = 0; q < nu; q++) {
            int in_o = 0;
            for (int p = 0; p < sub_n[O]; p++) if (sub_idx[O][p] == un[q]) in_o = 1;
            if (in_o) T[O].idx[T[O].rank++] = un[q];
        }
        if (T[O].rank > *max_rank) *max_rank = T[O].rank;
        if (T[L].rank > *max_rank) *max_rank = T[L].rank;
        if (T[R].rank > *max_rank) *max_rank = T[R].rank;
        size_t osz = (size_t)1 << T[O].rank;
        T[O].v = (elem *)malloc(sizeof(elem) * osz);
        if (!T[O].v) { rc = 5; break; }
        for (size_t i = 0; i < osz; i++) T[O].v[i] = el_zero();
        /* bit position of every union index inside L, R, O (or -1) */
        int pl[64], pr[64], po[64];
        for (int q = 0; q < nu; q++) {
            pl[q] = pr[q] = po[q] = -1;
            for (int p = 0; p < T[L].rank; p++) if (T[L].idx[p] == un[q]) pl[q] = p;
            for (int p = 0; p < T[R].rank; p++) if (T[R].idx[p] == un[q]) pr[q] = p;
            for (int p = 0; p < T[O].rank; p++) if (T[O].idx[p] == un[q]) po[q] = p;
        }
        /* out[proj_O] (+)= L[proj_L] (.) R[proj_R] over all joint assignments */
        for (uint64_t j = 0; j < ((uint64_t)1 << nu); j++) {
            size_t il = 0, ir = 0, io = 0;
            for (int q = 0; q < nu; q++) {
                size_t b = (size_t)((j >> q) & 1);
                if (pl[q] >= 0) il |= b << pl[q];
                if (pr[q] >= 0) ir |= b << pr[q];
                if (po[q] >= 0) io |= b << po[q];
            }
            T[O].v[io] = el_add(T[O].v[io], el_mul(T[L].v[il], T[R].v[ir]));
        }
        tensor_free(&T[L]); tensor_free(&T[R]);
    }
    if (!rc) {
        tensor *root = &T[total - 1];
        if (n_steps == 0) root = &T[0];
        if (root->rank != 0 && n_steps != 0) rc = 6;
        else {   /* a single input tensor (n_steps == 0) still has its index summed (Eq. 2) */
            elem acc = el_zero();
            for (size_t i = 0; i < ((size_t)1 << root->rank); i++) acc = el_add(acc, root->v[i]);
            write_out(acc, kind, energy, feasible, count4);
        }
    }
    for (int t = 0; t < total; t++) { tensor_free(&T[t]); free(sub_idx[t]); free(sub_cnt[t]); }
    free(T); free(occ_total); free(sub_idx); free(sub_cnt); free(sub_n); free(val);
    return rc;
}

/* ---- oracle-3: frontier (transfer-matrix) dynamic programme ------------------
 * Vertices are visited in `order` (all n of them, fixed ones included).  The
 * table is indexed by the bits of the frontier = visited free vertices that still
 * have an unvisited neighbour.  Visiting v multiplies in its vertex entry and the
 * bond entries to every visited neighbour, then sums out every frontier vertex
 * whose neighbours have all been visited.  No contraction tree is involved. */
int oracle_frontier_dp(int kind, int n, int m, const int32_t *eu, const int32_t *ev,
                       const int32_t *edge_w, const int32_t *vertex_w, const int32_t *order,
                       int n_fixed, const int32_t *fixed, const uint8_t *assign,
                       int64_t *energy, int32_t *feasible, uint64_t *count4, int32_t *max_frontier)
{
    int *val = (int *)malloc(sizeof(int) * (size_t)(n + 1));
    int *visited = (int *)calloc((size_t)(n + 1), sizeof(int));
    int *remaining = (int *)calloc((size_t)(n + 1), sizeof(int));   /* unvisited neighbours */
    for (int i = 0; i < n; i++) val[i] = -1;
    for (int j = 0; j < n_fixed; j++) val[fixed[j]] = assign[j] ? 1 : 0;
    for (int e = 0; e < m; e++) { remaining[eu[e]]++; remaining[ev[e]]++; }
    int fr[64], nfr = 0;          /* fr[p] = vertex at bit p */
    size_t sz = 1;
    elem *tab = (elem *)malloc(sizeof(elem));
    tab[0] = el_make(0, 1);
    int rc = 0; *max_frontier = 0;
    for (int step = 0; step < n && !rc; step++) {
        int v = order[step];
        if (v < 0 || v >= n || visited[v]) { rc = 2; break; }
        int isfree = val[v] < 0;
        if (isfree && nfr >= 30) { rc = 4; break; }
        size_t nsz = isfree ? sz * 2 : sz;
        elem *nt = (elem *)malloc(sizeof(elem) * nsz);
        if (!nt) { rc = 5; break; }
        /* visited neighbours of v: edge id, orientation, frontier bit or fixed value */
        int ne = 0, *ne_e = (int *)malloc(sizeof(int) * (size_t)(m + 1)), *ne_p = (int *)malloc(sizeof(int) * (size_t)(m + 1)),
            *ne_s = (int *)malloc(sizeof(int) * (size_t)(m + 1));
        for (int e = 0; e < m; e++) {
            int u = -1;
            if (eu[e] == v) u = ev[e]; else if (ev[e] == v) u = eu[e];
            if (u < 0 || !visited[u]) continue;
            ne_e[ne] = e; ne_s[ne] = val[u]; ne_p[ne] = -1;
            if (val[u] < 0) { int p; for (p = 0; p < nfr; p++) if (fr[p] == u) break; ne_p[ne] = p; }
            ne++;
        }
        #pragma omp parallel for schedule(static)
        for (size_t s = 0; s < sz; s++) {
            for (int x = 0; x < (isfree ? 2 : 1); x++) {
                int sv = isfree ? x : val[v];
                elem a = el_mul(tab[s], vertex_entry(kind, vw_of(kind, vertex_w, v), sv));
                for (int q = 0; q < ne; q++) {
                    int e = ne_e[q];
                    int su = ne_p[q] >= 0 ? (int)((s >> ne_p[q]) & 1) : ne_s[q];
                    a = el_mul(a, eu[e] == v ? bond_entry(kind, ew_of(edge_w, e), sv, su)
                                             : bond_entry(kind, ew_of(edge_w, e), su, sv));
                }
                nt[isfree ? (s | ((size_t)x << nfr)) : s] = a;
            }
        }
        free(ne_e); free(ne_p); free(ne_s);
        free(tab); tab = nt; sz = nsz;
        if (isfree) fr[nfr++] = v;
        visited[v] = 1;
        for (int e = 0; e < m; e++) { if (eu[e] == v) remaining[ev[e]]--; else if (ev[e] == v) remaining[eu[e]]--; }
        if (nfr > *max_frontier) *max_frontier = nfr;
        /* sum out finished frontier vertices */
        for (int p = nfr - 1; p >= 0; p--) {
            int u = fr[p];
            if (remaining[u] > 0) continue;
            size_t hs = sz / 2;
            elem *rt = (elem *)malloc(sizeof(elem) * hs);
            size_t low = ((size_t)1 << p) - 1;
            #pragma omp parallel for schedule(static)
            for (size_t s = 0; s < hs; s++) {
                size_t s0 = (s & low) | ((s & ~low) << 1);
                rt[s] = el_add(tab[s0], tab[s0 | ((size_t)1 << p)]);
            }
            free(tab); tab = rt; sz = hs;
            for (int q = p; q + 1 < nfr; q++) fr[q] = fr[q + 1];
            nfr--;
        }
    }
    if (!rc) { if (sz != 1) rc = 6; else write_out(tab[0], kind, energy, feasible, count4); }
    free(tab); free(val); free(visited); free(remaining);
    return rc;
}

/* ---- oracle-3, sparse form for MIS ("for MIS only independent frontier
 * states are stored") --------------------------------------------------------------------
 * Same vertex-by-vertex transfer as oracle_frontier_dp, but the table holds only the
 * frontier states that are independent sets (every other state is the zero element,
 * PAPER.md:55), as a list sorted by key.  key bit p = 1 <=> the frontier vertex in slot p
 * is in the set.  Visiting v: every state survives with v out; a state with no chosen
 * frontier neighbour of v also spawns (key | bit_v, e + w_v, c).  A frontier vertex whose
 * neighbours are all visited is summed out: its bit is cleared and equal keys are (+)-merged.
 * Both operations are merges of two key-sorted lists.  Handles frontiers of up to 64 vertices. */
typedef struct { uint64_t key; int64_t e; u256 c; } sstate;

int oracle_frontier_dp_mis_sparse(int n, int m, const int32_t *eu, const int32_t *ev,
                                  const int32_t *vertex_w, const int32_t *order,
                                  int n_fixed, const int32_t *fixed, const uint8_t *assign,
                                  int64_t *energy, int32_t *feasible, uint64_t *count4,
                                  int32_t *max_frontier, int64_t *max_states)
{
    int *val = (int *)malloc(sizeof(int) * (size_t)(n + 1));
    int *visited = (int *)calloc((size_t)(n + 1), sizeof(int));
    int *remaining = (int *)calloc((size_t)(n + 1), sizeof(int));
    int *slot = (int *)malloc(sizeof(int) * (size_t)(n + 1));
    for (int i = 0; i < n; i++) { val[i] = -1; slot[i] = -1; }
    for (int j = 0; j < n_fixed; j++) val[fixed[j]] = assign[j] ? 1 : 0;
    for (int e = 0; e < m; e++) { remaining[eu[e]]++; remaining[ev[e]]++; }
    uint64_t used = 0;            /* occupied slots */
    int nfr = 0, rc = 0;
    size_t sz = 1;
    sstate *tab = (sstate *)malloc(sizeof(sstate));
    tab[0].key = 0; tab[0].e = 0; tab[0].c = u256_from(1);
    *max_frontier = 0; *max_states = 1;
    for (int step = 0; step < n && !rc; step++) {
        int v = order[step];
        if (v < 0 || v >= n || visited[v]) { rc = 2; break; }
        int64_t w = vw_of(1, vertex_w, v);
        uint64_t nbmask = 0; int nb_fixed_in = 0;
        for (int e = 0; e < m; e++) {
            int u = -1;
            if (eu[e] == v) u = ev[e]; else if (ev[e] == v) u = eu[e];
            if (u < 0 || !visited[u]) continue;
            if (val[u] == 1) nb_fixed_in = 1;
            else if (val[u] < 0) nbmask |= 1ull << slot[u];
        }
        if (val[v] == 1) {
            /* forced in: states with a chosen neighbour die, the rest gain w */
            size_t k = 0;
            for (size_t s = 0; s < sz; s++)
                if (!nb_fixed_in && !(tab[s].key & nbmask)) { tab[k] = tab[s]; tab[k].e += w; k++; }
            sz = k;
        } else if (val[v] < 0) {
            if (nfr >= 64) { rc = 4; break; }
            int p = 0; while (used & (1ull << p)) p++;
            slot[v] = p; used |= 1ull << p; nfr++;
            if (!nb_fixed_in) {
                uint64_t bit = 1ull << p;
                sstate *nt = (sstate *)malloc(sizeof(sstate) * (2 * sz + 1));
                if (!nt) { rc = 5; break; }
                /* list "out" = tab as it is; list "in" = eligible states with the bit set; merge by key */
                size_t i = 0, j = 0, k = 0;
                while (j < sz && (tab[j].key & nbmask)) j++;
                while (i < sz || j < sz) {
                    if (j >= sz || (i < sz && tab[i].key < (tab[j].key | bit))) nt[k++] = tab[i++];
                    else {
                        nt[k] = tab[j]; nt[k].key |= bit; nt[k].e += w; k++;
                        j++; while (j < sz && (tab[j].key & nbmask)) j++;
                    }
                }
                free(tab); tab = nt; sz = k;
            }
        }
        visited[v] = 1;
        for (int e = 0; e < m; e++) { if (eu[e] == v) remaining[ev[e]]--; else if (ev[e] == v) remaining[eu[e]]--; }
        if (nfr > *max_frontier) *max_frontier = nfr;
        if ((int64_t)sz > *max_states) *max_states = (int64_t)sz;
        /* sum out every frontier vertex whose neighbours have all been visited */
        for (int u = 0; u < n && !rc; u++) {
            if (slot[u] < 0 || remaining[u] > 0) continue;
            uint64_t bit = 1ull << slot[u];
            sstate *nt = (sstate *)malloc(sizeof(sstate) * (sz + 1));
            if (!nt) { rc = 5; break; }
            size_t i = 0, j = 0, k = 0;     /* i walks states with the bit clear, j those with it set */
            while (i < sz && (tab[i].key & bit)) i++;
            while (j < sz && !(tab[j].key & bit)) j++;
            while (i < sz || j < sz) {
                uint64_t ki = i < sz ? tab[i].key : ~0ull, kj = j < sz ? (tab[j].key & ~bit) : ~0ull;
                if (i < sz && (j >= sz || ki < kj)) {
                    nt[k++] = tab[i];
                    i++; while (i < sz && (tab[i].key & bit)) i++;
                } else if (j < sz && (i >= sz || kj < ki)) {
                    nt[k] = tab[j]; nt[k].key = kj; k++;
                    j++; while (j < sz && !(tab[j].key & bit)) j++;
                } else {                    /* same key: (+) */
                    elem a = el_make(tab[i].e, 0), b = el_make(tab[j].e, 0);
                    a.c = tab[i].c; b.c = tab[j].c;
                    elem r = el_add(a, b);
                    nt[k].key = ki; nt[k].e = r.e; nt[k].c = r.c; k++;
                    i++; while (i < sz && (tab[i].key & bit)) i++;
                    j++; while (j < sz && !(tab[j].key & bit)) j++;
                }
            }
            free(tab); tab = nt; sz = k;
            used &= ~bit; slot[u] = -1; nfr--;
        }
    }
    if (!rc) {
        if (sz > 1) rc = 6;
        else if (sz == 0) write_out(el_zero(), 1, energy, feasible, count4);
        else { elem r = el_make(tab[0].e, 0); r.c = tab[0].c; write_out(r, 1, energy, feasible, count4); }
    }
    free(tab); free(val); free(visited); free(remaining); free(slot);
    return rc;
}

/* ---- raw counting-tropical GEMM, triple loop ---------------------------------
 * Inputs: energies int64, explicit zero flags, counts uint64 (taken as exact
 * integers).  Output counts are returned mod 2^64 (low limb) and, if Cc4 != NULL,
 * in full 256-bit form.  A is [B][M][K], Bm is [B][K][N], C is [B][M][N]. */
int oracle_gemm(int64_t B, int M, int N, int K,
                const int64_t *Ae, const uint8_t *Az, const uint64_t *Ac,
                const int64_t *Be, const uint8_t *Bz, const uint64_t *Bc,
                int64_t *Ce, uint8_t *Cz, uint64_t *Cc, uint64_t *Cc4)
{
    #pragma omp parallel for collapse(2) schedule(static)
    for (int64_t b = 0; b < B; b++)
        for (int i = 0; i < M; i++)
            for (int j = 0; j < N; j++) {
                elem acc = el_zero();
                for (int k = 0; k < K; k++) {
                    size_t ia = ((size_t)b * M + i) * K + k, ib = ((size_t)b * K + k) * N + j;
                    elem a = Az[ia] ? el_zero() : el_make(Ae[ia], Ac[ia]);
                    elem c = Bz[ib] ? el_zero() : el_make(Be[ib], Bc[ib]);
                    acc = el_add(acc, el_mul(a, c));
                }
                size_t ic = ((size_t)b * M + i) * N + j;
                Ce[ic] = acc.zero ? 0 : acc.e; Cz[ic] = (uint8_t)acc.zero; Cc[ic] = acc.zero ? 0 : acc.c.w[0];
                if (Cc4) for (int l = 0; l < 4; l++) Cc4[4 * ic + l] = acc.zero ? 0 : acc.c.w[l];
            }
    return 0;
}

/* ---- bit permutation: dst[pi(i)] = src[i], bit j of pi(i) = bit perm[j] of i -- */
int oracle_permute(int r, const int32_t *perm, int64_t B, const int32_t *src_e, const uint64_t *src_c,
                   int32_t *dst_e, uint64_t *dst_c)
{
    size_t n = (size_t)1 << r;
    for (int64_t b = 0; b < B; b++)
        for (size_t i = 0; i < n; i++) {
            size_t d = 0;
            for (int j = 0; j < r; j++) d |= ((i >> perm[j]) & 1) << j;
            dst_e[(size_t)b * n + d] = src_e[(size_t)b * n + i];
            dst_c[(size_t)b * n + d] = src_c[(size_t)b * n + i];
        }
    return 0;
}

/* ---- region bound (reading A15) ---------------------
 * bound = sum over terms with every endpoint fixed of their exact value
 *       + sum over regions j of  max over the free vertices of R_j of the terms
 *         whose support lies inside R_j u F and touches R_j
 *       + sum over every remaining term of its largest entry compatible with the
 *         fixed endpoints.
 * MIS: a term's entries are 0 or w; an infeasible fixed pair gives "zero" (infeasible=1).
 * The result is in max-plus units (Ising: an upper bound on -H). */
int oracle_region_bound(int kind, int n, int m, const int32_t *eu, const int32_t *ev,
                        const int32_t *edge_w, const int32_t *vertex_w,
                        int n_regions, const int32_t *region_offsets, const int32_t *region_vertices,
                        int n_fixed, const int32_t *fixed, const uint8_t *assign,
                        int64_t *bound, int32_t *infeasible)
{
    int *val = (int *)malloc(sizeof(int) * (size_t)(n + 1));
    int *reg = (int *)malloc(sizeof(int) * (size_t)(n + 1));
    for (int i = 0; i < n; i++) { val[i] = -1; reg[i] = -1; }
    for (int j = 0; j < n_fixed; j++) val[fixed[j]] = assign[j] ? 1 : 0;
    for (int j = 0; j < n_regions; j++)
        for (int p = region_offsets[j]; p < region_offsets[j + 1]; p++) {
            int v = region_vertices[p];
            if (val[v] >= 0) continue;            /* fixed vertices are not free region members */
            if (reg[v] >= 0) { free(val); free(reg); return 2; }   /* regions must be disjoint */
            reg[v] = j;
        }
    int64_t tot = 0; *infeasible = 0;
    /* (a) fully fixed terms, (c) uncovered terms */
    for (int e = 0; e < m; e++) {
        int u = eu[e], v = ev[e];
        int fu = val[u] >= 0, fv = val[v] >= 0;
        if (fu && fv) {
            elem x = bond_entry(kind, ew_of(edge_w, e), val[u], val[v]);
            if (x.zero) *infeasible = 1; else tot += x.e;
            continue;
        }
        /* covered iff every free endpoint lies in one and the same region */
        int ru = fu ? -2 : reg[u], rv = fv ? -2 : reg[v];
        int covered = (ru != -1 && rv != -1) && (ru == -2 || rv == -2 || ru == rv);
        if (covered) continue;
        int64_t best = 0; int have = 0;
        for (int su = 0; su < 2; su++) for (int sv = 0; sv < 2; sv++) {
            if (fu && su != val[u]) continue;
            if (fv && sv != val[v]) continue;
            elem x = bond_entry(kind, ew_of(edge_w, e), su, sv);
            if (x.zero) continue;
            if (!have || x.e > best) { best = x.e; have = 1; }
        }
        tot += best;
    }
    for (int i = 0; i < n; i++) {
        if (val[i] >= 0) { tot += vertex_entry(kind, vw_of(kind, vertex_w, i), val[i]).e; continue; }
        if (reg[i] >= 0) continue;
        /* uncovered free vertex: largest vertex entry; MIS: 0 if a neighbour is fixed to 1 */
        int64_t e0 = vertex_entry(kind, vw_of(kind, vertex_w, i), 0).e, e1 = vertex_entry(kind, vw_of(kind, vertex_w, i), 1).e;
        int allow1 = 1;
        if (kind == 1)
            for (int e = 0; e < m; e++) {
                int o = -1; if (eu[e] == i) o = ev[e]; else if (ev[e] == i) o = eu[e];
                if (o >= 0 && val[o] == 1) allow1 = 0;
            }
        tot += (allow1 && e1 > e0) ? e1 : e0;
    }
    /* (b) regions: exact max over their free vertices */
    for (int j = 0; j < n_regions && !*infeasible; j++) {
        int fv[32], nf = 0;
        for (int p = region_offsets[j]; p < region_offsets[j + 1]; p++)
            if (val[region_vertices[p]] < 0) { if (nf >= 26) { free(val); free(reg); return 4; } fv[nf++] = region_vertices[p]; }
        if (nf == 0) continue;
        int have = 0; int64_t best = 0;
        for (uint32_t x = 0; x < (1u << nf); x++) {
            for (int q = 0; q < nf; q++) val[fv[q]] = (int)((x >> q) & 1);
            int64_t s = 0; int ok = 1;
            for (int q = 0; q < nf; q++) s += vertex_entry(kind, vw_of(kind, vertex_w, fv[q]), val[fv[q]]).e;
            for (int e = 0; e < m && ok; e++) {
                int u = eu[e], v = ev[e];
                int inu = val[u] >= 0 && reg[u] == j, inv = val[v] >= 0 && reg[v] == j;
                if (!inu && !inv) continue;                 /* does not touch R_j */
                if (val[u] < 0 || val[v] < 0) continue;     /* other endpoint free and outside */
                if (!inu && reg[u] >= 0) continue;          /* other endpoint in another region: uncovered */
                if (!inv && reg[v] >= 0) continue;
                elem t = bond_entry(kind, ew_of(edge_w, e), val[u], val[v]);
                if (t.zero) ok = 0; else s += t.e;
            }
            if (ok && (!have || s > best)) { best = s; have = 1; }
        }
        for (int q = 0; q < nf; q++) val[fv[q]] = -1;
        if (!have) *infeasible = 1; else tot += best;
    }
    *bound = tot;
    free(val); free(reg);
    return 0;
}

/* ---- Eq. 4: rho = sum_T max(0, log2|T| - log2 T_target) -------- */
int64_t oracle_rho(int n_tensors, const int32_t *log2_sizes, int32_t log2_target)
{
    int64_t r = 0;
    for (int i = 0; i < n_tensors; i++) if (log2_sizes[i] > log2_target) r += log2_sizes[i] - log2_target;
    return r;
}
