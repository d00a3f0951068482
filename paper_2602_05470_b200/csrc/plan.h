// plan.h -- host-side planner of the BBTN contraction engine (plain C++, no CUDA).
//
// For one fixed-set signature F (Eq. 3) the planner turns
// (graph, SSA tree) into a list of device steps: which input tensors K1 builds,
// how every pairwise contraction (Eq. 2 evaluated pairwise) maps
// onto index classes  g = I_L n I_R n I_O,  K = (I_L n I_R) \ I_O,
// M = I_L \ I_R,  N = I_R \ I_L,  which bit permutations K2 must apply, which
// K3 variant runs, and where every tensor lives in the device arena.
// All tensor dimensions are 2, so a rank-r tensor is 2^r elements and a layout
// is the list of index labels per bit of the linear element index.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace bbtn {

struct Problem {
  int kind = 0;                       // 0 Ising, 1 MIS
  int n = 0, m = 0;
  std::vector<int32_t> eu, ev, ew, vw;  // ew/vw always materialised (defaults applied)
  std::vector<int32_t> tree_l, tree_r;  // empty = derive per signature
  int64_t max_elements = (int64_t)1 << 28;
  int64_t energy_range = (int64_t)1 << 28;   // sum of |couplings| + |fields/weights|: bounds every finite energy of every tensor
  uint32_t flags = 0;
};

// One input tensor as K1 must build it.
struct InputRec {
  int32_t type;        // 0 bond, 1 vertex
  int32_t u, v;        // vertex ids (v = -1 for vertex tensors)
  int32_t w;           // J_ij or h_i / w_i
  int32_t fu, fv;      // column of u / v inside `assign`, or -1 when free
  int32_t su, sv;      // 1 if the free index u / v occurs in no other tensor: summed inside K1 (reading A7)
  int32_t bu, bv;      // bit position of u / v in the emitted tensor, -1 if absent
  int32_t rank;        // rank of the emitted tensor (0 => folded into offset[b])
  int32_t variant;     // depends on the assignment
  int64_t offset;      // element offset in the arena (rank > 0)
};

enum StepKind : int32_t { STEP_ABSORB = 0, STEP_REDUCE = 1, STEP_PERMUTE = 2, STEP_GEMM = 3 };

// A device launch.  Offsets are element offsets into the arena; batch strides are 0 for
// leaf-invariant tensors (contracted once, broadcast to every leaf).
struct Step {
  int32_t kind = 0;
  int32_t variant = 0;          // 1: runs for every leaf, 0: once
  // ABSORB / REDUCE: out[o] = (+)_k A[fa(o) + ka(k)] (.) B[fb(o) + kb(k)]
  int32_t rO = 0, nK = 0;
  uint32_t addA[32] = {0}, addB[32] = {0};   // per output bit
  uint32_t kA[32] = {0}, kB[32] = {0};       // per contracted bit
  // tensor locations: element offset inside the variant arena (per-leaf units; the real
  // offset is off * B, the tensor is [B][2^rank]) or inside the invariant arena.
  int64_t offA = 0, offB = 0, offC = 0;
  int32_t vA = 0, vB = 0, vC = 0;            // 1 = lives in the variant arena
  int32_t rA = 0, rB = 0;                    // operand ranks (batch stride = vX ? 2^rX : 0)
  // PERMUTE: dst[pi(i)] = src[i], bit j of pi(i) = bit perm[j] of i   (offA -> offC, rank rO)
  int32_t perm[32] = {0};
  // GEMM: A [g][k][m], B [g][k][n] -> C [g][m][n]   (log2 sizes)
  int32_t lg = 0, lm = 0, ln = 0, lk = 0;
  // upper bound on log2(count + 1) of BOTH operands (inputs hold counts 0/1, each (.) adds the operands' bounds,
  // each (+) over 2^k terms adds k): lets K3 pick its narrow count modes inside a tree; 64 = no useful bound
  int32_t count_bits = 64;
  // every count of operand B is 0 or 1 (B is built from input tensors only, nothing summed yet): the count product is
  // then the count of A -- the streaming kernels skip the multiply and the load of B's counts.  (A zero element of B has
  // energy -inf, which makes the term lose against any finite term or be canonicalised away, whatever count it carries.)
  int32_t b_unit = 0;
  // local slicing (make_local_plan): an operand that is a view of a stored tensor starts at
  // off + sum_j x_j * slice[j], x = the current assignment of the segment's fixed indices
  int32_t n_slice = 0;
  int32_t xA = 0, xB = 0;                    // operand is such a view: it lives in the invariant arena, sliced per batch entry
  uint32_t sliceA[24] = {0}, sliceB[24] = {0};
  double fma = 0;               // tropical FMAs of this launch per batch entry
  double bytes = 0;             // algorithmic bytes per batch entry (12 B per element moved)
};

struct Plan {
  std::vector<int32_t> fixed;
  std::vector<InputRec> inputs;          // all n_in inputs in ABI order
  std::vector<int32_t> scalar_inputs;    // ids of inputs folded into offset[b]
  std::vector<Step> steps;
  int64_t result_offset = -1;            // rank-0 result tensor, -1 if the network is all scalars
  int32_t result_variant = 0;
  int64_t arena_variant_elems = 0;       // per-leaf elements (multiply by B)
  int64_t arena_invariant_elems = 0;
  int32_t max_rank = 0;
  int64_t rho = 0;
  double fma_variant = 0, fma_invariant = 0;
  double bytes_variant = 0, bytes_invariant = 0;
  int32_t n_nodes = 0, n_variant_nodes = 0;
  // filled when make_plan is asked to (want_labels): the index labels of every launched node's
  // output tensor, in step order -- the tensors Eq. 4 sums over (used by the branching driver)
  std::vector<std::vector<int32_t>> node_labels;
};

// ---- local slicing (BBTN on sub-networks) -------------------------------------------------------
// The tree is walked in SSA order and cut into SEGMENTS.  A segment whose tensors fit T_target runs once.
// A segment that holds tensors above T_target gets a LOCAL fixed set F (indices that are summed inside the
// segment): the segment is contracted once per assignment x of F (Eq. 3, applied to the sub-TN)
// with every tensor carrying an index of F cut down to its x-slice, and the one tensor that leaves the
// segment and depends on F is the (+) over x of the slices' results -- for every state of the segment's
// boundary the (energy, count) of its interior (the counting form of the boundary-equivalence principle,
// PAPER.md:67; reading A16).  Tensors that enter a sliced segment are stored in full and read
// through strided views, so nothing outside the segment is ever contracted twice.
struct LocalSeg {
  std::vector<int32_t> fixed;            // F; empty = the segment runs once
  int32_t step_begin = 0, step_end = 0;  // range in Plan::steps
  std::vector<int32_t> list_var;         // inputs K1 builds for every slice (they touch F; rank > 0 under F)
  std::vector<int32_t> list_inv;         // inputs of the stretch that do not depend on F: built once per launch sequence
  std::vector<int32_t> list_scalar;      // inputs that are scalars under F: their product is the slice's offset
  int32_t acc_rank = -1;                 // sliced segments: the F-dependent tensor leaving the segment ...
  int64_t acc_off = 0, tmp_off = 0;      // ... is accumulated at acc_off (invariant arena) from the per-slice results at tmp_off (variant arena)
  int32_t max_rank = 0;
  double fma = 0, bytes = 0;             // per slice (bytes include the accumulation pass)
};
struct LocalPlan {
  Plan plan;                             // inputs (each under its segment's F), all steps, arena size, result offset
  std::vector<LocalSeg> segs;
  int32_t cap_rank = 0;
  double fma_total = 0, bytes_total = 0; // over all slices of all segments (infeasible slices included)
  double n_slices = 0;                   // sum over segments of 2^|F|
  int32_t max_fixed = 0, n_sliced_segs = 0;
};
// P must carry a tree (tree_l/tree_r non-empty).  cap_rank = log2 T_target.  Returns 0 or a status; ESHAPE when a
// segment cannot be brought under T_target (needs more than 24 fixed indices, or the tree joins two sliced parts).
int make_local_plan(const Problem &P, int cap_rank, LocalPlan &out, std::string &err);

// Returns 0 or a bbtn_status value; err receives the message.
// force_mode: 0 = automatic, 1 = never use the tiled GEMM path, 2 = use it wherever |K| >= 1.
// enforce_cap: fail with ESHAPE when a tensor exceeds P.max_elements (otherwise only rho records it).
// single_arena: place every tensor in the leaf-variant arena (one-leaf plans of the branching driver,
// which reuse one device buffer across different fixed sets).  want_labels: fill Plan::node_labels.
int make_plan(const Problem &P, const std::vector<int32_t> &fixed, int force_mode, bool enforce_cap,
              Plan &out, std::string &err, bool single_arena = false, bool want_labels = false);

// Elimination-order tree for the network with `fixed` sliced out (used when the caller gave no tree).
void derive_tree(const Problem &P, const std::vector<int32_t> &fixed,
                 std::vector<int32_t> &tl, std::vector<int32_t> &tr);

// Building blocks of derive_tree, also used by the local-branching driver to pick its tree: bucket elimination along a
// vertex order, and two order heuristics (plan.cpp).
void elimination_tree_for_order(const Problem &P, const std::vector<int32_t> &fixed, const std::vector<int> &order,
                                std::vector<int32_t> &tl, std::vector<int32_t> &tr, int &width, double &cost);
std::vector<int> min_degree_order(const Problem &P, const std::vector<int32_t> &fixed);
std::vector<int> mincut_sweep_order(const Problem &P, int delta, int window, const std::vector<int> *base = nullptr);

}  // namespace bbtn
