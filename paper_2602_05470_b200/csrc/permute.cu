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
  CT *sh_c = reinterpret_cast<CT *>(smem);
  int32_t *sh_e = reinterpret_cast<int32_t *>(smem + sizeof(CT) * tile);
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
      sh_c[i] = src_c[sbase + s];
    }
    __syncthreads();
    // scatter: thread index bits enumerate the tile in destination order
    for (int i = threadIdx.x; i < tile; i += blockDim.x) {
      uint32_t d = 0; int j = 0;
      for (int q = 0; q < p.nt; q++) if ((i >> q) & 1) { int tb = p.dperm[q]; j |= 1 << tb; d += p.tile_dst[tb]; }
      dst_e[dbase + d] = sh_e[j];
      dst_c[dbase + d] = sh_c[j];
    }
    __syncthreads();
  }
}

}  // namespace

void launch_permute(int rank, const int32_t *perm, int64_t batch, const int32_t *src_e, const void *src_c,
                    int32_t *dst_e, void *dst_c, int ring, cudaStream_t st) {
  // inverse: where does source bit s land
  int inv[32];
  for (int j = 0; j < rank; j++) inv[perm[j]] = j;
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
  const size_t csz = ring == 0 ? 8 : 4;
  const size_t smem = ((size_t)1 << nt) * (csz + 4);
  if (ring == 0)
    permute_kernel<uint64_t><<<grid, 256, smem, st>>>(p, src_e, (const uint64_t *)src_c, dst_e, (uint64_t *)dst_c);
  else
    permute_kernel<uint32_t><<<grid, 256, smem, st>>>(p, src_e, (const uint32_t *)src_c, dst_e, (uint32_t *)dst_c);
}

}  // namespace bbtn
