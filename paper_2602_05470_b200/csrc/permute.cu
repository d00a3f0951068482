// permute.cu -- K2: batched bit-permutation of a (energy, count) tensor (sm_100a).
//
//   dst[b][pi(i)] = src[b][i],   bit j of pi(i) = bit perm[j] of i.
//
// All tensor dimensions are 2, so "moving contracted legs to GEMM order" (north_star) is a
// permutation of the bits of the linear index.  The kernel splits the index bits into
//   * a LOW group  that is contiguous in the SOURCE  (the TS lowest source bits),
//   * a LOW group  that is contiguous in the DESTINATION (the TD lowest destination bits),
//   * the remaining bits, which only select which tile a CTA works on.
// A CTA gathers the tile spanned by (source-low u destination-low) bits with coalesced,
// vectorised reads along the source-low bits, stages it in shared memory and writes it with
// coalesced stores along the destination-low bits.  HBM-bound: 24 B per element (12 in + 12 out).
#include <type_traits>

#include "kernels.h"
#include "ring.cuh"

namespace bbtn {
namespace {

struct PermArgs {
  int rank;
  int nt;                 // number of tile bits (|source-low u destination-low|)
  int ns;                 // source-low bits (a prefix of the tile bits in source order)
  uint32_t tile_src[16];  // tile bit q  -> source offset
  uint32_t tile_dst[16];  // tile bit q  -> destination offset, enumerated in SOURCE-friendly order
  int dperm[16];          // destination-friendly enumeration: write index bit q -> tile bit
  uint32_t outer_src[32]; // outer bit q -> source offset
  uint32_t outer_dst[32]; // outer bit q -> destination offset
  int n_outer;
  int64_t batch;
};

template <class CT>
__global__ void __launch_bounds__(256) permute_kernel(PermArgs p, const int32_t *__restrict__ src_e,
                                                      const CT *__restrict__ src_c, int32_t *__restrict__ dst_e,
                                                      CT *__restrict__ dst_c) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int tile = 1 << p.nt;
  constexpr bool HC = !std::is_same<CT, NoCount>::value;            // search mode moves the energy plane alone
  CT *sh_c = reinterpret_cast<CT *>(smem);
  int32_t *sh_e = reinterpret_cast<int32_t *>(smem + (HC ? sizeof(CT) : 0) * tile);
  const int64_t n_tiles = ((int64_t)1 << p.n_outer) * p.batch;
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    const int64_t b = t >> p.n_outer;
    const uint32_t o = (uint32_t)(t & (((int64_t)1 << p.n_outer) - 1));
    uint32_t so = 0, d_o = 0;
    for (int q = 0; q < p.n_outer; q++) if ((o >> q) & 1u) { so += p.outer_src[q]; d_o += p.outer_dst[q]; }
    const int64_t sbase = (b << p.rank) + so, dbase = (b << p.rank) + d_o;
    // gather: thread index bits enumerate the tile in source order (low bits contiguous in src)
    for (int i = threadIdx.x; i < tile; i += blockDim.x) {
      uint32_t s = 0;
      for (int q = 0; q < p.nt; q++) if ((i >> q) & 1) s += p.tile_src[q];
      sh_e[i] = src_e[sbase + s];
      if constexpr (HC) sh_c[i] = src_c[sbase + s];
    }
    __syncthreads();
    // scatter: thread index bits enumerate the tile in destination order
    for (int i = threadIdx.x; i < tile; i += blockDim.x) {
      uint32_t d = 0; int j = 0;
      for (int q = 0; q < p.nt; q++) if ((i >> q) & 1) { int tb = p.dperm[q]; j |= 1 << tb; d += p.tile_dst[tb]; }
      dst_e[dbase + d] = sh_e[j];
      if constexpr (HC) dst_c[dbase + d] = sh_c[j];
    }
    __syncthreads();
  }
}

// ---- vectorised form (rank >= 4): 16-byte global accesses on both sides -----------------------
// Tile bits 0,1 (source enumeration) are source bits 0,1 and the two lowest destination bits are tile
// bits too, so a thread reads 4 source-contiguous elements per vector and writes 4 destination-contiguous
// ones.  Shared-memory address of tile index i is i ^ X(i), X XOR-linear in the bits of i and built on the
// host so that the lanes of the scatter phase (which walk destination bits 2..6) land on distinct banks
// where possible; X only uses bits >= 5 as sources and bits 2..4 as targets, which keeps the 16-byte
// staging stores contiguous and conflict-free.
struct PermVecArgs {
  int rank, nt, n_outer;
  int64_t batch;
  uint32_t tile_src[12];   // tile bit q (source enumeration) -> source offset
  uint32_t tile_dst[12];   // tile bit q -> destination offset
  uint32_t swz[12];        // tile bit q -> XOR contribution to the shared-memory address (includes 1<<q)
  int dperm[12];           // destination enumeration bit q -> tile bit
  uint32_t outer_src[32], outer_dst[32];
};

template <class CT> struct Vec4;
template <> struct Vec4<uint64_t> {
  ulonglong2 a, b;
  // global side: one 32-byte access per thread (LDG/STG.E.256 on sm_100) instead of two half-filled sectors per instruction
  __device__ __forceinline__ void gload(const uint64_t *p) {
    asm("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(a.x), "=l"(a.y), "=l"(b.x), "=l"(b.y) : "l"(p));
  }
  __device__ __forceinline__ void gstore(uint64_t *p) const {
    asm volatile("st.global.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(a.x), "l"(a.y), "l"(b.x), "l"(b.y));
  }
  __device__ __forceinline__ void load(const uint64_t *p) { a = *reinterpret_cast<const ulonglong2 *>(p); b = *reinterpret_cast<const ulonglong2 *>(p + 2); }
  __device__ __forceinline__ void store(uint64_t *p) const { *reinterpret_cast<ulonglong2 *>(p) = a; *reinterpret_cast<ulonglong2 *>(p + 2) = b; }
  __device__ __forceinline__ void set(int u, uint64_t v) { if (u == 0) a.x = v; else if (u == 1) a.y = v; else if (u == 2) b.x = v; else b.y = v; }
};

template <> struct Vec4<NoCount> {
  __device__ __forceinline__ void load(const NoCount *) {}
  __device__ __forceinline__ void store(NoCount *) const {}
  __device__ __forceinline__ void gload(const NoCount *) {}
  __device__ __forceinline__ void gstore(NoCount *) const {}
};

template <class CT>
__global__ void __launch_bounds__(256, 2) permute_vec_kernel(PermVecArgs p, const int32_t *__restrict__ src_e,
                                                          const CT *__restrict__ src_c, int32_t *__restrict__ dst_e,
                                                          CT *__restrict__ dst_c) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int tile = 1 << p.nt, nvec = tile >> 2;
  constexpr bool HC = !std::is_same<CT, NoCount>::value;
  CT *sh_c = reinterpret_cast<CT *>(smem);
  int32_t *sh_e = reinterpret_cast<int32_t *>(smem + (HC ? sizeof(CT) : 0) * tile);
  constexpr int VPT = 4;                               // vectors per thread at nt = 12
  // per-thread tables: vector v = threadIdx.x + 256*k
  uint32_t s_off[VPT], s_adr[VPT], d_off[VPT], d_adr[VPT], u_adr[4];
#pragma unroll
  for (int k = 0; k < VPT; k++) {
    const uint32_t i = (uint32_t)(threadIdx.x + 256 * k) << 2;
    uint32_t so = 0, sa = 0, dd = 0, da = 0;
    for (int q = 2; q < p.nt; q++)
      if ((i >> q) & 1u) {
        so += p.tile_src[q]; sa ^= p.swz[q];
        const int tb = p.dperm[q];
        dd += p.tile_dst[tb]; da ^= p.swz[tb];
      }
    s_off[k] = so; s_adr[k] = sa; d_off[k] = dd; d_adr[k] = da;
  }
#pragma unroll
  for (int u = 0; u < 4; u++) u_adr[u] = ((u & 1) ? p.swz[p.dperm[0]] : 0u) ^ ((u & 2) ? p.swz[p.dperm[1]] : 0u);

  const int64_t n_tiles = ((int64_t)1 << p.n_outer) * p.batch;
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    const int64_t b = t >> p.n_outer;
    const uint32_t o = (uint32_t)(t & (((int64_t)1 << p.n_outer) - 1));
    uint32_t so = 0, d_o = 0;
    for (int q = 0; q < p.n_outer; q++) if ((o >> q) & 1u) { so += p.outer_src[q]; d_o += p.outer_dst[q]; }
    const int64_t sbase = (b << p.rank) + so, dbase = (b << p.rank) + d_o;
    // gather: 4 source-contiguous elements per vector, all loads issued before the staging stores
    int4 ve[VPT]; Vec4<CT> vc[VPT];
#pragma unroll
    for (int k = 0; k < VPT; k++)
      if (threadIdx.x + 256 * k < nvec) {
        ve[k] = *reinterpret_cast<const int4 *>(src_e + sbase + s_off[k]);
        vc[k].gload(src_c + sbase + s_off[k]);
      }
#pragma unroll
    for (int k = 0; k < VPT; k++)
      if (threadIdx.x + 256 * k < nvec) {
        *reinterpret_cast<int4 *>(sh_e + s_adr[k]) = ve[k];
        vc[k].store(sh_c + s_adr[k]);
      }
    __syncthreads();
    // scatter: 4 destination-contiguous elements per vector
#pragma unroll
    for (int k = 0; k < VPT; k++)
      if (threadIdx.x + 256 * k < nvec) {
        int32_t e[4]; Vec4<CT> c;
#pragma unroll
        for (int u = 0; u < 4; u++) { const uint32_t a = d_adr[k] ^ u_adr[u]; e[u] = sh_e[a]; if constexpr (HC) c.set(u, sh_c[a]); }
        *reinterpret_cast<int4 *>(dst_e + dbase + d_off[k]) = make_int4(e[0], e[1], e[2], e[3]);
        c.gstore(dst_c + dbase + d_off[k]);
      }
    __syncthreads();
  }
}

}  // namespace

namespace {
inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

// vectorised path; returns false when the shape or alignment does not allow it
bool launch_permute_vec(int rank, const int32_t *perm, const int *inv, int64_t batch, const int32_t *src_e, const void *src_c,
                        int32_t *dst_e, void *dst_c, int ring, cudaStream_t st) {
  if (rank < 4 || !aligned16(src_e) || !aligned16(src_c) || !aligned16(dst_e) || !aligned16(dst_c)) return false;
  if (ring_count_bytes(ring) == 8 && ((reinterpret_cast<uintptr_t>(src_c) | reinterpret_cast<uintptr_t>(dst_c)) & 31)) return false;   // 32-byte count vectors
  PermVecArgs p;
  p.rank = rank; p.batch = batch;
  const int LOW = rank < 5 ? rank : 5;
  const int NT_MAX = 12;
  bool in_tile[32] = {false};
  int tile_bits[12]; int nt = 0;                  // tile bits as SOURCE bit numbers, source-low first
  for (int s = 0; s < LOW; s++) { tile_bits[nt++] = s; in_tile[s] = true; }
  for (int j = 0; j < LOW; j++) { int s = perm[j]; if (!in_tile[s]) { tile_bits[nt++] = s; in_tile[s] = true; } }
  // grow alternately along the source and the destination so both sides keep long contiguous runs
  for (int s = LOW, j = LOW; nt < NT_MAX && (s < rank || j < rank);) {
    while (s < rank && in_tile[s]) s++;
    if (s < rank && nt < NT_MAX) { tile_bits[nt++] = s; in_tile[s] = true; }
    while (j < rank && in_tile[perm[j]]) j++;
    if (j < rank && nt < NT_MAX) { tile_bits[nt++] = perm[j]; in_tile[perm[j]] = true; }
  }
  p.nt = nt;
  for (int q = 0; q < nt; q++) { p.tile_src[q] = 1u << tile_bits[q]; p.tile_dst[q] = 1u << inv[tile_bits[q]]; p.swz[q] = 1u << q; }
  int order[12];
  for (int q = 0; q < nt; q++) order[q] = q;
  for (int a = 0; a < nt; a++)
    for (int b2 = a + 1; b2 < nt; b2++)
      if (inv[tile_bits[order[b2]]] < inv[tile_bits[order[a]]]) { int t = order[a]; order[a] = order[b2]; order[b2] = t; }
  for (int q = 0; q < nt; q++) p.dperm[q] = order[q];
  // swizzle: the scatter lanes walk tile bits dperm[2..6]; fold those that are >= 5 into free bank bits 2..4
  bool low_used[5] = {false, false, false, false, false};
  for (int q = 2; q < 7 && q < nt; q++) if (order[q] < 5) low_used[order[q]] = true;
  int targets[3], n_t = 0;
  for (int b2 = 2; b2 < 5; b2++) if (!low_used[b2]) targets[n_t++] = b2;
  for (int q = 2, k = 0; q < 7 && q < nt; q++)
    if (order[q] >= 5) {
      const int tb = n_t > 0 ? targets[k % n_t] : 2 + (k % 3);
      p.swz[order[q]] |= 1u << tb; k++;
    }
  p.n_outer = 0;
  for (int s = 0; s < rank; s++) if (!in_tile[s]) { p.outer_src[p.n_outer] = 1u << s; p.outer_dst[p.n_outer] = 1u << inv[s]; p.n_outer++; }
  const int64_t n_tiles = ((int64_t)1 << p.n_outer) * batch;
  const int64_t cap = 148 * 8;
  const int grid = (int)(n_tiles < cap ? n_tiles : cap);
  const size_t csz = ring_count_bytes(ring);
  const size_t smem = ((size_t)1 << nt) * (csz + 4);
  if (csz == 8)                                           // mod 2^64, or both prime residues packed: pure data movement
    permute_vec_kernel<uint64_t><<<grid, 256, smem, st>>>(p, src_e, (const uint64_t *)src_c, dst_e, (uint64_t *)dst_c);
  else
    permute_vec_kernel<NoCount><<<grid, 256, smem, st>>>(p, src_e, (const NoCount *)src_c, dst_e, (NoCount *)dst_c);
  return true;
}
}  // namespace

void launch_permute(int rank, const int32_t *perm, int64_t batch, const int32_t *src_e, const void *src_c,
                    int32_t *dst_e, void *dst_c, int ring, cudaStream_t st) {
  // inverse: where does source bit s land
  int inv[32];
  for (int j = 0; j < rank; j++) inv[perm[j]] = j;
  if (launch_permute_vec(rank, perm, inv, batch, src_e, src_c, dst_e, dst_c, ring, st)) return;
  PermArgs p;
  p.rank = rank; p.batch = batch;
  const int LOW = rank < 5 ? rank : 5;            // 32 contiguous elements on each side
  bool in_tile[32] = {false};
  int tile_bits[16]; int nt = 0;                  // tile bits as SOURCE bit numbers
  for (int s = 0; s < LOW; s++) { tile_bits[nt++] = s; in_tile[s] = true; }
  p.ns = nt;
  for (int j = 0; j < LOW; j++) { int s = perm[j]; if (!in_tile[s]) { tile_bits[nt++] = s; in_tile[s] = true; } }
  // grow the tile (more source-contiguous bits) up to 2^11 elements to amortise the staging
  for (int s = LOW; s < rank && nt < 11; s++) if (!in_tile[s]) { tile_bits[nt++] = s; in_tile[s] = true; }
  p.nt = nt;
  for (int q = 0; q < nt; q++) { p.tile_src[q] = 1u << tile_bits[q]; p.tile_dst[q] = 1u << inv[tile_bits[q]]; }
  // destination-friendly enumeration: tile bits sorted by destination position
  int order[16];
  for (int q = 0; q < nt; q++) order[q] = q;
  for (int a = 0; a < nt; a++)
    for (int b2 = a + 1; b2 < nt; b2++)
      if (inv[tile_bits[order[b2]]] < inv[tile_bits[order[a]]]) { int t = order[a]; order[a] = order[b2]; order[b2] = t; }
  for (int q = 0; q < nt; q++) p.dperm[q] = order[q];
  p.n_outer = 0;
  for (int s = 0; s < rank; s++) if (!in_tile[s]) { p.outer_src[p.n_outer] = 1u << s; p.outer_dst[p.n_outer] = 1u << inv[s]; p.n_outer++; }
  const int64_t n_tiles = ((int64_t)1 << p.n_outer) * batch;
  const int64_t cap = 148 * 8;
  const int grid = (int)(n_tiles < cap ? n_tiles : cap);
  const size_t csz = ring_count_bytes(ring);
  const size_t smem = ((size_t)1 << nt) * (csz + 4);
  if (csz == 8)
    permute_kernel<uint64_t><<<grid, 256, smem, st>>>(p, src_e, (const uint64_t *)src_c, dst_e, (uint64_t *)dst_c);
  else
    permute_kernel<NoCount><<<grid, 256, smem, st>>>(p, src_e, (const NoCount *)src_c, dst_e, (NoCount *)dst_c);
}

}  // namespace bbtn
