/*
 * bbtn.h -- C ABI of the B200-native BBTN hot path.
 *
 * Exact contraction of counting-tropical tensor networks, batched over
 * branch-and-bound leaves (arxiv/paper_2602_05470; citations are PAPER.md:<line>).
 *
 *   element  = (energy, count)                       PAPER.md:53 (counting), :55 (zero = (inf,0))
 *   a (.) b  = (ea + eb, ca * cb)                    PAPER.md:49 (x (.) y = x + y)
 *   a (+) b  = the better energy; counts add on ties PAPER.md:49 (x (+) y = min(x,y)), :53
 *
 * The engine works in MAX-plus on negated Ising energies (the paper's min-sum
 * mirrored, reading A1); MIS is natively a maximisation.
 * Results are reported in the paper's units: Ising min H (Eq. 1),
 * MIS max set weight.
 *
 * Conventions that hold for EVERY entry point
 *   - plain C, no C++/torch types; all integers are fixed-width.
 *   - pointers are HOST pointers unless the parameter is documented "device" or the
 *     handle was built with BBTN_IO_DEVICE (then assign/energy/count/count_mod/bound
 *     of the batched calls are device pointers and the call is asynchronous on
 *     `cuda_stream`; with host pointers the call returns after the results landed).
 *   - the caller owns every array it passes; the library copies what it keeps.
 *     The handle owns all device memory, plans and CUDA graphs it creates.
 *   - every function returns a bbtn_status; on error no output is written and the
 *     message is available from bbtn_last_error(handle) (handle may be NULL for
 *     errors of handle-less calls: thread-local).
 *   - a handle is used by one host thread at a time.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).
 *   - integer arithmetic only: results are bit-identical across runs, trees,
 *     tilings and batch sizes.
 *   - there is NO CPU fallback: without a CUDA device every compute call returns
 *     BBTN_ECUDA.
 */
#ifndef BBTN_H_
#define BBTN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bbtn_handle bbtn_handle;            /* opaque, library-owned */

typedef enum { BBTN_ISING = 0, BBTN_MIS = 1 } bbtn_kind;

typedef enum {
  BBTN_OK = 0,
  BBTN_EINVAL = 1,     /* malformed argument (bad vertex id, duplicate fixed vertex, bad tree ...) */
  BBTN_ENOMEM = 2,     /* host or device allocation failed                                        */
  BBTN_ECUDA = 3,      /* CUDA runtime error or no device                                         */
  BBTN_ESHAPE = 4,     /* an intermediate would exceed max_elements_per_leaf (T_target)           */
  BBTN_ERANGE = 5      /* sum of |couplings| + |fields/weights| exceeds BBTN_ENERGY_LIMIT         */
} bbtn_status;

/* Energy of the semiring zero element ("(inf, 0)"); its count is 0.
 * Finite energies obey |e| <= BBTN_ENERGY_LIMIT, so NEG_INF + NEG_INF still fits an int32 and any
 * energy below -2^29 is canonicalised back to (BBTN_NEG_INF, 0) (reading A8).
 * Zero-ness is decided by the ENERGY, never by count == 0. */
#define BBTN_NEG_INF (-(1 << 30))
#define BBTN_ENERGY_LIMIT (1 << 28)

/* flags of bbtn_problem_desc.flags */
#define BBTN_COUNT_CRT 0x1u   /* also keep counts mod P1 and mod P2 (one more pass over the tree)  */
#define BBTN_IO_DEVICE 0x2u   /* batched calls take/return DEVICE pointers, asynchronous           */
#define BBTN_NO_GRAPH  0x4u   /* launch kernels one by one instead of replaying a CUDA graph       */
#define BBTN_FORCE_STREAMING 0x10u /* tuning/testing: never use the tiled GEMM + permute path          */
#define BBTN_FORCE_TILED     0x20u /* tuning/testing: permute + tiled GEMM wherever an index is summed */
#define BBTN_NO_FUSED        0x80u /* tuning/testing: never run a small network, or the small subtrees of a larger one, as a shared-memory launch (one CTA per leaf) */
#define BBTN_SEARCH_ONLY     0x40u /* ground-state SEARCH ("the tropical number inf for optimization problems",
                                      :81-91): plain max-plus, no count plane anywhere (4 B per element instead of 12);
                                      the batched calls and the solve drivers return the optimal energy only, every
                                      count output reads 0 and `count` may be NULL.  Excludes BBTN_COUNT_CRT */

#define BBTN_P1 2147483647u   /* 2^31 - 1  */
#define BBTN_P2 2147483629u   /* 2^31 - 19 */

/* The problem: a graph G=(V,E) with couplings/fields (Eq. 1) or vertex weights
 * (MWIS), plus a contraction tree.  Input tensors are numbered
 *   0 .. n_edges-1                      the bond tensor of edge e on indices (s_u, s_v)
 *   n_edges .. n_edges+n_vertices-1     the vertex tensor of vertex i on index (s_i)
 * and step t of the SSA tree contracts ids tree_l[t], tree_r[t] into id n_inputs + t; a complete
 * tree has n_inputs - 1 steps.  tree_l == NULL: the library derives an elimination-order tree
 * itself, per fixed set (results do not depend on the tree, only speed and width do). */
typedef struct {
  int32_t kind;                    /* bbtn_kind                                                  */
  int32_t n_vertices, n_edges;
  const int32_t *edge_u, *edge_v;  /* [n_edges], 0 <= u != v < n_vertices, no duplicate edges    */
  const int32_t *edge_w;           /* Ising: integer J_ij per edge (NULL = all +1). MIS: ignored */
  const int32_t *vertex_w;         /* Ising: integer h_i (NULL = no field). MIS: w_i (NULL = 1)  */
  int32_t n_steps;                 /* 0 with tree_l == NULL, else n_edges + n_vertices - 1       */
  const int32_t *tree_l, *tree_r;  /* [n_steps] or NULL                                          */
  int64_t max_elements_per_leaf;   /* T_target of Eq. 4, in ELEMENTS, <= 2^32; 0 = 2^28 */
  uint32_t flags;
} bbtn_problem_desc;

/* What the planner derived for one fixed-set signature and batch size. */
typedef struct {
  int32_t n_nodes;            /* pairwise contraction steps that launch work                       */
  int32_t n_variant_nodes;    /* of which depend on the leaf assignment (the rest run once)        */
  int32_t max_rank;           /* log2 of the largest tensor of one leaf (contraction width)        */
  int32_t n_gemm_tiled, n_absorb, n_permute, n_trace;   /* kernel launches per count ring, by kind */
  int64_t rho;                /* Eq. 4 with T_target = max_elements_per_leaf                       */
  double  fma_variant;        /* tropical FMAs per leaf in leaf-variant nodes                      */
  double  fma_invariant;      /* tropical FMAs in leaf-invariant nodes (once per call)             */
  double  bytes_per_call;     /* algorithmic bytes read+written by all kernels for this B          */
  int64_t workspace_bytes;    /* device memory the plan holds for this B                           */
  int32_t n_kernel_launches;  /* kernels one bbtn_contract_batch enqueues per count ring (K1..K4)  */
  int32_t reserved;
} bbtn_plan_info;

/* Build a handle: validates and copies the problem (graph, weights, tree).  Host only: device
 * tables and arenas are created by the first batched call.  Errors: EINVAL, ERANGE, ENOMEM. */
int bbtn_build(const bbtn_problem_desc *desc, bbtn_handle **out);

/* Contract one batch of B leaves that share the fixed set F (Eq. 3: the reduced TN
 * with s_{V_f} = x; "same topology but different contents").
 *   fixed_vertices [n_fixed]   distinct vertex ids (host, always)
 *   assign         [B][n_fixed] 0/1; 1 <=> sigma = +1 (Ising) / vertex in the set (MIS)
 *   energy         [B] int32   Ising: min over the free spins of H (fixed-fixed terms included),
 *                              so min_b energy[b] = E0;  MIS: max set weight given the assignment
 *   count          [B] uint64  number of optimal completions, mod 2^64
 *   count_mod      [B][2] uint32 residues mod BBTN_P1, BBTN_P2 (needs BBTN_COUNT_CRT), or NULL
 * An infeasible leaf (MIS: two adjacent vertices fixed to 1) returns energy BBTN_NEG_INF, count 0.
 * n_fixed = 0 with B = 1 is the unbranched contraction (assign may be NULL).
 * Steps run on the device: K1 construct, K2 permute, K3 counting-tropical GEMM, K4 trace.
 * Errors: EINVAL, ESHAPE, ENOMEM, ECUDA. */
int bbtn_contract_batch(bbtn_handle *h,
                        const int32_t *fixed_vertices, int32_t n_fixed,
                        const uint8_t *assign, int64_t B,
                        int32_t *energy, uint64_t *count, uint32_t *count_mod,
                        void *cuda_stream);

/* Plan (or look up) the signature without running it. */
int bbtn_plan_query(bbtn_handle *h, const int32_t *fixed_vertices, int32_t n_fixed, int64_t B,
                    bbtn_plan_info *info);

/* Local bounds for pruning ("evaluating local energy contributions over a subset
 * of variables R"; reading A15).  Regions are disjoint vertex sets in CSR form
 * (region_offsets [n_regions+1], region_vertices); fixed vertices listed in a region are ignored;
 * a region may hold at most 20 free vertices.
 *   bound[b] = exact value of every term whose endpoints are all fixed
 *            + sum_j max over the free vertices of R_j of the terms inside R_j u F touching R_j
 *            + for every other term its largest entry compatible with the fixed endpoints
 * in the units of energy[]: Ising bound[b] <= energy[b] (a LOWER bound on min H), MIS
 * bound[b] >= energy[b].  Infeasible leaf: BBTN_NEG_INF (MIS).  One warp per (leaf, region) (K5). */
int bbtn_region_bound(bbtn_handle *h,
                      const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions,
                      const int32_t *fixed_vertices, int32_t n_fixed,
                      const uint8_t *assign, int64_t B,
                      int32_t *bound, void *cuda_stream);

/* bbtn_region_bound for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same bound, same kernels (K5), but
 *   - `assign` [B][n_fixed] and `bound` [B] are DEVICE pointers whatever the handle's flags say;
 *   - the per-(leaf, region) maxima go to a file-scope device array of BBTN_REGION_BOUND_STATIC_MAX_ITEMS int32
 *     (4 MiB, held by every GPU that loads the library until the process exits) instead of a handle buffer:
 *     B * max(n_regions, 1) beyond that is refused with BBTN_ESHAPE;
 *   - the K5 tables of (regions, fixed_vertices) must already be cached in the handle by an earlier ordinary
 *     bbtn_region_bound call with the same regions and fixed vertices (set-up; the cache holds 64 signatures): if they
 *     are not, the call fails with BBTN_EINVAL instead of building (and allocating) them.
 * The call allocates and frees no device memory, copies nothing, does not synchronise: it launches the two K5 kernels
 * on `cuda_stream` and returns.  B = 0 is the set-up call: it checks the tables and resolves the array's device address
 * for the current device (also done by the first real call on each device) and launches nothing.
 * Every call on a GPU shares the one array, which keeps the last call's contents (every entry a call reads it has
 * written first, so nothing is cleared): calls that OVERLAP on the GPU (different streams) race and return garbage;
 * calls on one stream are safe.  Errors: EINVAL, ESHAPE, ECUDA. */
#define BBTN_REGION_BOUND_STATIC_MAX_ITEMS (1 << 20)
int bbtn_region_bound_static(bbtn_handle *h,
                             const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions,
                             const int32_t *fixed_vertices, int32_t n_fixed,
                             const uint8_t *assign_device, int64_t B,
                             int32_t *bound_device, void *cuda_stream);

/* Host branch-and-bound driver (global pruning :67; S6): depth-first
 * over `branch_vertices` in the given order, `chunk` levels at a time; every partial assignment is
 * bounded with bbtn_region_bound and discarded iff its bound is strictly worse than the incumbent
 * (ties kept, reading A14); surviving full assignments are contracted in batches of <= max_batch
 * with bbtn_contract_batch and (+)-accumulated.
 *   incumbent_hint: energy (reported units) of some feasible configuration known to the caller,
 *   used only to prune earlier; BBTN_NEG_INF = none.  A hint better than the true optimum
 *   makes the search return (BBTN_NEG_INF, 0).
 *   energy/count/count_mod: the exact optimum over ALL configurations; stats[0..3] = nodes
 *   generated, pruned, leaves contracted, contract calls.  Host pointers only. */
int bbtn_solve_bb(bbtn_handle *h,
                  const int32_t *branch_vertices, int32_t n_branch, int32_t chunk,
                  const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions,
                  int64_t max_batch, int32_t incumbent_hint, int32_t use_pruning,
                  int32_t *energy, uint64_t *count, uint32_t *count_mod, int64_t *stats,
                  void *cuda_stream);

/* BBTN proper: non-uniform branching driven by the memory-overflow measure
 *   rho(T) = sum over the tensors of the contraction tree of max(0, log2|T| - log2 T_target)   (Eq. 4)
 * on the handle's contraction tree (the caller's, else the library's tree of the unsliced network).
 * Each branching takes the free vertex v that minimises the branching factor gamma, the root of
 * gamma^rho(T) = sum_i gamma^rho(T_i), over the rules
 *   MIS:   { v = 0 } , { v = 1 and every free neighbour of v = 0 }        Ising: { s_v = 0 } , { s_v = 1 }
 * (complete and orthogonal; the paper's rule search and inference rules are in its missing
 * supplement, reading A23).  A branch with rho = 0 whose arena fits mem_budget_bytes is a leaf:
 * its fixed indices are deleted from the tree, it is contracted by K1..K4 on the device (one plan per leaf,
 * device buffers reused) and the leaf results are (+)-accumulated.  Leaves have DIFFERENT fixed sets
 * ("different subsets of R are fixed across different branches").
 *   log2_target       log2 T_target in ELEMENTS, 1..32 (the paper runs 2^31)
 *   mem_budget_bytes  device bytes one leaf may use; 0 = 94 % of the free device memory
 *   max_leaves        give up with BBTN_ESHAPE beyond this many leaves; 0 = unlimited
 *   energy/count/count_mod  as bbtn_solve_bb;  stats[0..3] = branching nodes, leaves, largest |F|, rho of the root
 *   work[0..1] = tropical FMAs, algorithmic bytes summed over the leaves (planner totals)
 * Host pointers only.  Errors: EINVAL, ESHAPE, ENOMEM, ECUDA. */
int bbtn_solve_branching(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes, int64_t max_leaves,
                         int32_t *energy, uint64_t *count, uint32_t *count_mod, int64_t *stats, double *work,
                         void *cuda_stream);

/* The same branching without contracting anything (host only, no device needed): writes the leaves in CSR
 * form -- leaf i fixes leaf_vertices[leaf_offsets[i] .. leaf_offsets[i+1]) to leaf_values[...] -- when the three
 * arrays are non-NULL (capacities cap_leaves + 1 offsets, cap_entries vertices/values; EINVAL if too small),
 * and stats/work as above.  mem_budget_bytes = 0 means no memory limit here. */
int bbtn_branching_leaves(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes, int64_t max_leaves,
                          int64_t cap_leaves, int64_t cap_entries, int64_t *leaf_offsets, int32_t *leaf_vertices,
                          uint8_t *leaf_values, int64_t *stats, double *work);

/* BBTN on sub-networks ("local branching"; PAPER.md:65-69, :67 boundary equivalence; readings A16, A25).
 * The contraction tree (the caller's, else the library's tree of the unsliced network) is walked in order.  Where
 * every tensor fits T_target = 2^log2_target elements the steps run once.  A stretch of the tree whose tensors
 * overflow T_target is a sub-TN with open legs: it is decomposed by fixing a LOCAL set F of variables that are all
 * summed inside it, chosen greedily to bring Eq. 4's overflow rho of the stretch to zero; every branch (assignment
 * of F) is contracted by K1..K3 on slices of the stored tensors that enter the stretch, and the tensor that leaves
 * it is the (+) over the branches -- per boundary state the (energy, count) of the interior.  Nothing
 * outside a stretch is contracted more than once, so the cost is sum over stretches of 2^|F| x (its own cost)
 * instead of 2^(sum |F|) x (the whole tree).  Branches are pruned before contraction: infeasible
 * ones (MIS: two adjacent vertices of F set), and, when regions (as for bbtn_region_bound) and an incumbent are
 * given, those whose K5 bound is strictly worse than the incumbent (ties kept, reading A14).
 *   incumbent_hint  energy (reported units) of a feasible configuration known to the caller; BBTN_NEG_INF = none
 *   mem_budget_bytes  0 = 94 % of the free device memory; the threshold is lowered until the arena fits
 * The branches of one stretch share one plan (one signature F): the survivors are contracted as BATCHES, as many at
 * a time as fit the memory budget (the batch axis of K1 and K3; slices of the stored tensors are addressed per batch
 * entry from the branch's assignment row), so a stretch with many small branches costs a few launch sequences.
 *   stats[0..11] = stretches, sliced stretches, branches planned (sum of 2^|F|), branches contracted, branches
 *                  infeasible, branches pruned by bound, largest |F|, largest tensor rank, arena bytes, kernel launches,
 *                  branches in flight per launch sequence, launch sequences
 *   work[0..3]   = tropical FMAs and algorithmic bytes over all planned branches (12 B per element read or written),
 *                  the same two over the branches actually contracted
 * Host pointers only.  Errors: EINVAL, ESHAPE (a stretch needs more than 24 fixed variables, or the tree joins two
 * overflowing parts so that no local set exists), ENOMEM, ECUDA. */
int bbtn_solve_local(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes,
                     const int32_t *region_offsets, const int32_t *region_vertices, int32_t n_regions,
                     int32_t incumbent_hint,
                     int32_t *energy, uint64_t *count, uint32_t *count_mod, int64_t *stats, double *work,
                     void *cuda_stream);

/* A hint for the library's tree search (only used when the handle was built WITHOUT a tree): `order` [n_vertices] is
 * a permutation of the vertices, e.g. a sweep of the caller's geometry in another direction.  bbtn_solve_local derives
 * its candidate trees (nested-minimum-cut sweeps, reading A26) from the vertex-id order, from every hinted
 * order and from each of them reversed, plans all of them and keeps the cheapest.  Results never depend on it.
 * Host only.  Errors: EINVAL (not a permutation). */
int bbtn_add_sweep_order(bbtn_handle *h, const int32_t *order);

/* The plan bbtn_solve_local would run, without running it (host only, no device): stats / work as above
 * (the run-time entries 3, 4, 5, 9, 10, 11 and work[2..3] are zero).  mem_budget_bytes = 0 means no memory limit here. */
int bbtn_local_plan_query(bbtn_handle *h, int32_t log2_target, int64_t mem_budget_bytes, int64_t *stats, double *work);

/* Host-side (+) over leaf results in reported units (Eq. 3's outer sum; "the final
 * result is obtained by summing the contractions of each branch"): keeps the best
 * energy (Ising: lowest, MIS: highest), adds the counts of the leaves that attain it (mod 2^64,
 * and mod P1/P2 when count_mod != NULL).  Infeasible leaves (BBTN_NEG_INF) are neutral; if all n
 * are infeasible (or n == 0) the result is (BBTN_NEG_INF, 0).  Part of S6 (plain C++, no device):
 * bbtn_solve_bb uses it per batch, a multi-process driver uses it across ranks.
 *   kind: bbtn_kind; energy/count [n]; count_mod [n][2] or NULL; out_count_mod [2] or NULL. */
int bbtn_oplus_combine(int32_t kind, int64_t n, const int32_t *energy, const uint64_t *count,
                       const uint32_t *count_mod, int32_t *out_energy, uint64_t *out_count,
                       uint32_t *out_count_mod);

/* CRT recombination of the three count residues of BBTN_COUNT_CRT mode (reading A9): 2^64, BBTN_P1 and
 * BBTN_P2 are pairwise coprime, so (count mod 2^64, count mod P1, count mod P2) determine the count modulo
 * 2^64 * P1 * P2 (about 2^126).  out[0] = low 64 bits, out[1] = high 64 bits of that value; it IS the exact count
 * whenever the count is below 2^126.  Host only, no device.  Errors: EINVAL (null out, residue >= its prime). */
int bbtn_crt_combine(uint64_t count_mod_2_64, uint32_t count_mod_p1, uint32_t count_mod_p2, uint64_t out[2]);

/* Debug checks of caller promises (process-wide switch, default off; also switched on by the environment
 * variable BBTN_DEBUG_CHECKS=1 at load time).  When on, the raw GEMM entry points first verify ON THE DEVICE
 * that every operand count is below 2^count_bits (for count_bits < 64) and that every operand energy is either
 * exactly BBTN_NEG_INF or below 2^energy_bits in magnitude (within +-BBTN_ENERGY_LIMIT for energy_bits >= 29), synchronise, and return BBTN_EINVAL without launching K3
 * if a promise is broken.  Returns the previous setting. */
int bbtn_set_debug_checks(int32_t on);

/* Raw batched counting-tropical GEMM (K3 alone; the config-4 sweep):
 *   C[b,m,n] = (+)_k A[b,m,k] (.) B[b,k,n]
 * ALL pointers are DEVICE pointers.  Row-major: A [batch][M][K], B [batch][K][N], C [batch][M][N];
 * stride* are the ELEMENT distances between consecutive batch entries (0 = operand shared by the
 * whole batch).  Energies int32: the zero element must be passed in its canonical form (BBTN_NEG_INF, count 0),
 * finite energies obey |e| <= BBTN_ENERGY_LIMIT; outputs are canonical, so results can be fed back in.  Other
 * energies are a broken promise (sums could wrap): undefined results, caught by bbtn_set_debug_checks.
 * Counts uint64 mod 2^64.  M, N, K >= 1, any size (ragged tiles are handled); the launch is refused with
 * BBTN_ESHAPE if it would need more than 2^31-1 thread blocks.
 * count_bits in 1..64: upper bound on log2(count+1) of BOTH operands that the caller guarantees (64 = no
 * promise; <= 32 selects the 32x32->64 multiply path, small values 32-bit accumulators).
 * energy_bits in 1..32: the caller guarantees |e| < 2^energy_bits for every FINITE operand energy (32 = no promise
 * beyond BBTN_ENERGY_LIMIT).  energy_bits <= 11 together with count_bits <= 32 selects the packed form: 16-bit
 * energies, two outputs per instruction, with 32-bit accumulators where 2 * count_bits + ceil(log2 K) <= 32, a
 * 31-bit running sum plus carry register for count_bits <= 13, and 64-bit accumulators otherwise.
 * A broken promise gives wrong results silently unless bbtn_set_debug_checks is on.  The result never depends on
 * which form ran.  Asynchronous on cuda_stream. */
int bbtn_tropical_gemm_batched(int64_t batch, int32_t M, int32_t N, int32_t K,
                               const int32_t *Ae, const uint64_t *Ac,
                               const int32_t *Be, const uint64_t *Bc,
                               int32_t *Ce, uint64_t *Cc,
                               int64_t strideA, int64_t strideB, int64_t strideC,
                               int32_t count_bits, int32_t energy_bits, void *cuda_stream);

/* Same operation with HOST pointers (the end-to-end form of the config-4 sweep): the operands are
 * copied to library-owned device staging buffers, K3 runs, C is copied back and the call returns after
 * the results landed.  The batch flows in chunks through three internal streams ordered after
 * `cuda_stream`, so with PINNED host memory the PCIe copies of one chunk overlap the GEMM of another.
 * On BBTN_ECUDA during the copy-back the contents of Ce/Cc are unspecified. */
int bbtn_tropical_gemm_batched_host(int64_t batch, int32_t M, int32_t N, int32_t K,
                                    const int32_t *Ae, const uint64_t *Ac,
                                    const int32_t *Be, const uint64_t *Bc,
                                    int32_t *Ce, uint64_t *Cc,
                                    int64_t strideA, int64_t strideB, int64_t strideC,
                                    int32_t count_bits, int32_t energy_bits, void *cuda_stream);

/* K3 of the SEARCH mode alone (PAPER.md:55 "the tropical number inf for optimization problems", :81-91; Eq. 2
 * evaluated pairwise, :51, :57, in the max-plus semiring without counts):
 *   C[b][m][n] = max_k ( A[b][m][k] + B[b][k][n] ),   energies int32, row-major, DEVICE pointers,
 * strides in elements between batch entries (0 = operand shared by the whole batch).  The zero element is
 * BBTN_NEG_INF: any energy below -2^29 is read as zero, a sum that involves a zero is zero, outputs are canonical
 * (exactly BBTN_NEG_INF).  Finite energies must lie within +-BBTN_ENERGY_LIMIT.
 *   energy_bits  1..32, the caller's PROMISE that every finite operand energy is below 2^energy_bits in magnitude;
 *                <= 11 selects the packed form (two 16-bit add-max per integer instruction), anything else the
 *                32-bit form; results do not depend on it when the promise holds (checked on the device when
 *                bbtn_set_debug_checks is on).
 * Asynchronous on cuda_stream.  Errors: EINVAL, ESHAPE (more than 2^31-1 thread blocks), ECUDA. */
int bbtn_maxplus_gemm_batched(int64_t batch, int32_t M, int32_t N, int32_t K,
                              const int32_t *A, const int32_t *B, int32_t *C,
                              int64_t strideA, int64_t strideB, int64_t strideC,
                              int32_t energy_bits, void *cuda_stream);

/* Raw batched bit permutation (K2 alone): dst[b][pi(i)] = src[b][i] for i in [0, 2^rank), where
 * bit j of pi(i) is bit perm[j] of i (perm is a HOST array, a permutation of 0..rank-1).
 * Both planes (int32 energies, uint64 counts) move; DEVICE pointers; asynchronous. */
int bbtn_permute_batched(int32_t rank, const int32_t *perm, int64_t batch,
                         const int32_t *src_e, const uint64_t *src_c,
                         int32_t *dst_e, uint64_t *dst_c, void *cuda_stream);

/* Integer-pipe microbenchmarks (register-only, no memory traffic) that define the ALU roofline of
 * K3.  which: 0 = IADD3 chain, 1 = IMNMX chain, 2 = fused add-max
 * (VIADDMNMX), 3 = IMAD chain, 4 = mixed 3-operand IADD3+IMAD (both pipes), 7 / 8 = mixed two-operand
 * IADD:IMAD at 1:1 / 2:1, 9 / 10 = the instruction stream of K3's inner loop (fused add-max, add, tie
 * compare, predicated IMAD, operand LDS.128 from a broadcast table) at 2 / 4+ warps per SM sub-partition;
 * 5, 6 = earlier op-mix kernels (kept for comparison, not used by bench.py); 11..15 = issue rates of the building
 * blocks of the packed and 64-bit forms with operands that change every round: 11 VIADDMNMX.S16x2, 12 HSETP2 + SEL,
 * 13 ISETP + SEL, 14 IMAD.WIDE with 64-bit accumulate, 15 the packed pair (add-max16x2, add, HSETP2, 2 predicated IMAD).
 * Runs `iters` unrolled rounds on every SM; returns elapsed milliseconds (CUDA events) and the
 * number of lane-operations (which <= 4, 7, 8), tropical FMAs (5, 6, 9, 10) or lane-rounds (11..15) executed. */
int bbtn_int32_microbench(int32_t which, int32_t iters, double *milliseconds, double *operations,
                          void *cuda_stream);

void bbtn_destroy(bbtn_handle *h);                    /* NULL is a no-op */
const char *bbtn_last_error(const bbtn_handle *h);    /* valid until the next call on h / this thread */
const char *bbtn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BBTN_H_ */
