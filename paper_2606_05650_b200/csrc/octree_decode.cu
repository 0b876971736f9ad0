// Decoder-side position coder (section 2.3, Alg. A.2 / A.3): occupancy bytes -> Morton codes of
// the occupied voxels -> integer coordinates.
//
// count -> prefix-sum -> scatter, as in the paper, except that the popcount prefix sum is taken ONCE over
// the whole breadth-first stream instead of once per level: with G = exclusive scan of popcount(byte) over
// all S bytes, the children of the p-th node of level d start at position G[off_d + p] - G[off_d] of
// L_{d+1} (off_d = stream offset of level d).  The level loop then only has to carry the codes down
// ((parent << 3) + i, Alg. A.3 l.4-9), one small launch per level, no per-level scan.
#include "common.cuh"

namespace gsnfs {

__device__ __forceinline__ uint32_t compact3(uint64_t x) {   // every third bit -> 21 contiguous bits
  x &= 0x1249249249249249ull;
  x = (x | (x >> 2)) & 0x10c30c30c30c30c3ull;
  x = (x | (x >> 4)) & 0x100f00f00f00f00full;
  x = (x | (x >> 8)) & 0x001f0000ff0000ffull;
  x = (x | (x >> 16)) & 0x001f00000000ffffull;
  x = (x | (x >> 32)) & 0x1fffffull;
  return (uint32_t)x;
}

// One thread per node of level d (Alg. A.3).  LAST: children are leaves -> also emit (x, y, z).
template <bool LAST>
__global__ void __launch_bounds__(256) expand_children_kernel(
    const uint64_t* __restrict__ L_d, const uint8_t* __restrict__ occ_d, const uint32_t* __restrict__ G_d,
    uint32_t m_d, uint32_t m_next, uint64_t* __restrict__ L_next, uint32_t* __restrict__ xyz,
    gsnfs_counts* __restrict__ counts) {
  const uint32_t p = blockIdx.x * 256 + threadIdx.x;
  if (p >= m_d) return;
  const uint32_t occ = occ_d[p];
  const uint32_t g0 = G_d[0];
  uint32_t w = G_d[p] - g0;
  const uint32_t cnt = __popc(occ);
  bool bad = (occ == 0u) || (w + cnt > m_next);
  if (p == m_d - 1 && w + cnt != m_next) bad = true;          // sum popcount(level d) != |L_{d+1}|  [O12]
  if (bad) atomicOr(&counts->status, 1u);
  if (w + cnt > m_next) return;
  const uint64_t base = L_d[p] << 3;
  uint32_t bits = occ;
  while (bits) {
    const int i = __ffs(bits) - 1;
    bits &= bits - 1;
    const uint64_t code = base + (uint64_t)i;
    if (L_next) L_next[w] = code;
    if (LAST) {
      xyz[3 * (size_t)w + 0] = compact3(code);
      xyz[3 * (size_t)w + 1] = compact3(code >> 1);
      xyz[3 * (size_t)w + 2] = compact3(code >> 2);
    }
    ++w;
  }
}

__global__ void decode_init_kernel(uint64_t* L0, gsnfs_counts* counts, uint32_t nv, uint32_t occ_bytes,
                                   uint32_t status) {
  L0[0] = 0;                         // implicit root code (Alg. A.2 l.2)
  counts->n_voxels = nv;
  counts->occ_bytes = occ_bytes;
  counts->status = status;
  counts->reserved = 0;
}

int run_octree_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_occ, uint64_t occ_bytes,
                      const uint32_t* level_sizes, int depth, uint32_t* d_voxel_xyz, uint64_t* d_voxel_keys,
                      gsnfs_counts* d_counts) {
  const uint32_t nv = level_sizes[depth];
  uint64_t sum = 0;
  for (int d = 0; d < depth; ++d) sum += level_sizes[d];
  uint32_t status = 0;
  if (nv == 0) {
    if (occ_bytes != 0) status = 1;
    GSNFS_KERNEL(ctx, st, "decode_init");
    decode_init_kernel<<<1, 1, 0, st>>>(ctx->dec_keys_a, d_counts, 0, (uint32_t)occ_bytes, status);
    GSNFS_LAUNCH_CHECK(ctx, st);
    return GSNFS_OK;
  }
  if (sum != occ_bytes || level_sizes[0] != 1) status = 1;    // header inconsistent with the stream [O12]
  for (int d = 0; d <= depth; ++d)
    if (level_sizes[d] > ctx->max_points) return GSNFS_E_CAPACITY;
  if (occ_bytes + 1 > ctx->occ_cap) return GSNFS_E_CAPACITY;
  GSNFS_KERNEL(ctx, st, "decode_init");
  decode_init_kernel<<<1, 1, 0, st>>>(ctx->dec_keys_a, d_counts, nv, (uint32_t)occ_bytes, status);
  GSNFS_LAUNCH_CHECK(ctx, st);
  if (status) return GSNFS_OK;        // reported through d_counts->status; nothing decoded
  int rc = run_scan_popc8(ctx, st, d_occ, ctx->dec_scan, (uint32_t)occ_bytes);
  if (rc != GSNFS_OK) return rc;
  uint64_t* cur = ctx->dec_keys_a;
  uint64_t* nxt = ctx->dec_keys_b;
  uint64_t off = 0;
  for (int d = 0; d < depth; ++d) {
    const uint32_t m_d = level_sizes[d], m_next = level_sizes[d + 1];
    const uint32_t grid = (m_d + 255) / 256;
    GSNFS_KERNEL(ctx, st, "expand_children");
    if (d == depth - 1) {
      expand_children_kernel<true><<<grid, 256, 0, st>>>(cur, d_occ + off, ctx->dec_scan + off, m_d, m_next,
                                                         d_voxel_keys, d_voxel_xyz, d_counts);
    } else {
      expand_children_kernel<false><<<grid, 256, 0, st>>>(cur, d_occ + off, ctx->dec_scan + off, m_d, m_next, nxt,
                                                          nullptr, d_counts);
    }
    GSNFS_LAUNCH_CHECK(ctx, st);
    off += m_d;
    uint64_t* t = cur; cur = nxt; nxt = t;
  }
  return GSNFS_OK;
}

}  // namespace gsnfs
