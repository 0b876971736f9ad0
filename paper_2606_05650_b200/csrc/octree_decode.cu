// Decoder-side position coder (section 2.3, Alg. A.2 / A.3): occupancy bytes -> Morton codes of
// the occupied voxels -> integer coordinates.
//
// count -> prefix-sum -> scatter, as in the paper, with two changes for launch/latency economy:
//  * the popcount prefix sum is taken ONCE over the whole breadth-first stream instead of once per level:
//    with G[n] = sum of popcount(byte m) over m < n, the children of stream node n are the nodes
//    G[n] + 1 ... of the breadth-first numbering (root = 0), i.e. positions G[n] + 1 - off[d+1] ... of L_{d+1};
//  * everything runs in one cooperative kernel, and because G is known for every node up front, one thread
//    can carry a code down TWO levels ((parent << 3) + i, Alg. A.3 l.4-9, applied twice) between grid-wide
//    barriers: ceil(J/2) barriers instead of 4J kernel launches.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

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

constexpr int kDecPrefixCap = 8192;   // tile sums whose prefix fits in shared memory (16 Mi stream bytes)

struct DecLevels {
  uint32_t size[GSNFS_MAX_DEPTH + 2];   // |L_d|, d = 0..J
  uint32_t off[GSNFS_MAX_DEPTH + 2];    // stream offset of level d (off[J] = S)
  int depth;
};

__device__ __forceinline__ void emit_leaf(uint64_t code, uint32_t pos, uint64_t* __restrict__ keys_out,
                                          uint32_t* __restrict__ xyz) {
  if (keys_out) keys_out[pos] = code;
  xyz[3 * (size_t)pos + 0] = compact3(code);
  xyz[3 * (size_t)pos + 1] = compact3(code >> 1);
  xyz[3 * (size_t)pos + 2] = compact3(code >> 2);
}

__device__ __forceinline__ uint32_t popc8x8(uint2 a) {
  return __popc(a.x) + __popc(a.y);
}

__global__ void __launch_bounds__(256) octree_decode_kernel(const uint8_t* __restrict__ occ, uint32_t S, DecLevels lv,
                                                            uint32_t* __restrict__ G, uint32_t* __restrict__ tile_sums,
                                                            uint64_t* ka, uint64_t* kb, uint32_t* __restrict__ xyz,
                                                            uint64_t* __restrict__ keys_out,
                                                            gsnfs_counts* __restrict__ counts,
                                                            unsigned long long* __restrict__ tstamp) {
  cg::grid_group grid = cg::this_grid();
  int ts = 0;
#define GSNFS_STAMP() do { if (blockIdx.x == 0 && threadIdx.x == 0 && ts < kRahtMaxPhases + 2) tstamp[ts] = globaltimer_ns(); ++ts; } while (0)
  GSNFS_STAMP();
  __shared__ uint32_t s_w[9];
  __shared__ uint32_t s_pre[kDecPrefixCap];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int J = lv.depth;
  if (blockIdx.x == 0 && tid == 0) {
    counts->n_voxels = lv.size[J];
    counts->occ_bytes = S;
    counts->status = 0;
    counts->reserved = 0;
    ka[0] = 0;                                   // implicit root code (Alg. A.2 l.2)
  }
  // ---- 1. G = exclusive scan of popcount(byte) over the stream (tile sums, barrier, down-sweep)
  const uint32_t ntile = (S + kScanTile - 1) / kScanTile;
  for (uint32_t t = blockIdx.x; t < ntile; t += gridDim.x) {
    const uint32_t i0 = t * kScanTile + tid * 8;
    uint32_t s = 0;
    if (i0 + 8 <= S) {
      s = popc8x8(*reinterpret_cast<const uint2*>(occ + i0));
    } else {
      for (uint32_t k = i0; k < S && k < i0 + 8; ++k) s += __popc((unsigned)occ[k]);
    }
    s = __reduce_add_sync(0xffffffffu, s);
    if (lane == 0) s_w[warp] = s;
    __syncthreads();
    if (tid == 0) {
      uint32_t tot = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) tot += s_w[k];
      tile_sums[t] = tot;
    }
    __syncthreads();
  }
  grid.sync();
  GSNFS_STAMP();
  // exclusive prefix of the tile sums, once per CTA, kept in shared memory (fallback: summed per tile)
  const bool pre_in_smem = ntile <= (uint32_t)kDecPrefixCap;
  if (pre_in_smem) {
    uint32_t carry = 0;
    for (uint32_t b0 = 0; b0 < ntile; b0 += 256) {
      const uint32_t k = b0 + tid;
      const uint32_t v = k < ntile ? __ldcg(tile_sums + k) : 0u;
      uint32_t tot;
      const uint32_t ex = block_excl_scan_256(v, s_w, &tot);
      if (k < ntile) s_pre[k] = carry + ex;
      carry += tot;
    }
    __syncthreads();
  }
  for (uint32_t t = blockIdx.x; t < ntile; t += gridDim.x) {
    uint32_t base = 0;
    if (pre_in_smem) {
      base = s_pre[t];
    } else {
      uint32_t part = 0;
      for (uint32_t k = tid; k < t; k += 256) part += __ldcg(tile_sums + k);
      part = __reduce_add_sync(0xffffffffu, part);
      if (lane == 0) s_w[warp] = part;
      __syncthreads();
#pragma unroll
      for (int k = 0; k < 8; ++k) base += s_w[k];
      __syncthreads();
    }
    const uint32_t i0 = t * kScanTile + tid * 8;
    uint32_t v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = 0;
    if (i0 + 8 <= S) {
      const uint2 a = *reinterpret_cast<const uint2*>(occ + i0);
#pragma unroll
      for (int k = 0; k < 4; ++k) { v[k] = __popc((a.x >> (8 * k)) & 0xffu); v[4 + k] = __popc((a.y >> (8 * k)) & 0xffu); }
    } else {
#pragma unroll
      for (int k = 0; k < 8; ++k) if (i0 + k < S) v[k] = __popc((unsigned)occ[i0 + k]);
    }
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
    uint32_t run = base + block_excl_scan_256(s, s_w, nullptr);
    if (i0 + 8 <= S) {
      uint4 a, b;
      a.x = run; run += v[0]; a.y = run; run += v[1]; a.z = run; run += v[2]; a.w = run; run += v[3];
      b.x = run; run += v[4]; b.y = run; run += v[5]; b.z = run; run += v[6]; b.w = run; run += v[7];
      *reinterpret_cast<uint4*>(G + i0) = a;
      *reinterpret_cast<uint4*>(G + i0 + 4) = b;
      if (i0 + 8 == S) G[S] = run;               // G has S + 1 entries; G[S] = total
    } else {
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        if (i0 + k <= S) G[i0 + k] = run;
        run += v[k];
      }
    }
  }
  grid.sync();
  GSNFS_STAMP();
  // ---- 2. carry the codes down, two levels per barrier.  While the levels are tiny ("top" steps) only
  // CTA 0 works and a block barrier is enough; the first large step is preceded by one grid barrier.
  const uint32_t gtid = blockIdx.x * 256 + tid, gstride = gridDim.x * 256;
  uint64_t* cur = ka;
  uint64_t* nxt = kb;
  int d = 0;
  bool top = true;
  while (d < J) {
    const bool two = d + 2 <= J;
    const uint32_t m_d = lv.size[d], m_1 = lv.size[d + 1];
    const uint32_t off_d = lv.off[d], off_1 = lv.off[d + 1];
    const uint32_t m_2 = two ? lv.size[d + 2] : 0u, off_2 = two ? lv.off[d + 2] : 0u;
    const bool top_step = top && (two ? m_2 : m_1) <= 4096u;
    if (top && !top_step) {
      top = false;
      if (d > 0) grid.sync();
    }
    if (!top_step || blockIdx.x == 0) {
      const uint32_t pstride = top_step ? 256u : gstride;
      uint32_t p = top_step ? (uint32_t)tid : gtid;
      // software pipeline: the next node's byte / prefix / code are requested before this node is expanded
      uint32_t bits = 0, g = 0;
      unsigned long long key = 0;
      if (p < m_d) { bits = occ[off_d + p]; g = __ldcg(G + off_d + p); key = __ldcg(reinterpret_cast<const unsigned long long*>(cur) + p); }
      while (p < m_d) {
        const uint32_t pn = p + pstride;
        uint32_t bits_n = 0, g_n = 0;
        unsigned long long key_n = 0;
        if (pn < m_d) { bits_n = occ[off_d + pn]; g_n = __ldcg(G + off_d + pn); key_n = __ldcg(reinterpret_cast<const unsigned long long*>(cur) + pn); }
        const uint32_t cnt = __popc(bits);
        const uint32_t cpos0 = g + 1u - off_1;                                     // position of the first child in L_{d+1}
        bool bad = (bits == 0u) || (cpos0 > m_1) || (cpos0 + cnt > m_1);
        if (p == m_d - 1 && cpos0 + cnt != m_1) bad = true;                        // sum popcount(level d) != |L_{d+1}| [O12]
        if (bad) {
          atomicOr(&counts->status, 1u);
        } else {
          const uint64_t base = (uint64_t)key << 3;
          if (!two) {
            uint32_t cpos = cpos0;
            while (bits) {
              const int i = __ffs(bits) - 1;
              bits &= bits - 1;
              const uint64_t ckey = base + (uint64_t)i;
              if (d + 1 == J) emit_leaf(ckey, cpos, keys_out, xyz); else nxt[cpos] = ckey;
              ++cpos;
            }
          } else {
            // the children are consecutive stream nodes: fetch all their bytes and prefix values at once
            const uint32_t c0 = off_1 + cpos0;                                     // stream index of the first child (d+1 < J)
            uint32_t b2[8], g2[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) {
              b2[r] = (uint32_t)r < cnt ? (uint32_t)occ[c0 + r] : 0u;
              g2[r] = (uint32_t)r < cnt ? __ldcg(G + c0 + r) : 0u;
            }
#pragma unroll
            for (int r = 0; r < 8; ++r) {
              if ((uint32_t)r < cnt) {
                const int i = __ffs(bits) - 1;
                bits &= bits - 1;
                const uint64_t ckey = base + (uint64_t)i;
                uint32_t bb = b2[r];
                const uint32_t cnt2 = __popc(bb);
                const uint32_t gpos0 = g2[r] + 1u - off_2;
                bool bad2 = (bb == 0u) || (gpos0 > m_2) || (gpos0 + cnt2 > m_2);
                if (cpos0 + r == m_1 - 1 && gpos0 + cnt2 != m_2) bad2 = true;
                if (bad2) {
                  atomicOr(&counts->status, 1u);
                } else {
                  const uint64_t base2 = ckey << 3;
                  uint32_t gpos = gpos0;
                  while (bb) {
                    const int j = __ffs(bb) - 1;
                    bb &= bb - 1;
                    const uint64_t gkey = base2 + (uint64_t)j;
                    if (d + 2 == J) emit_leaf(gkey, gpos, keys_out, xyz); else nxt[gpos] = gkey;
                    ++gpos;
                  }
                }
              }
            }
          }
        }
        p = pn; bits = bits_n; g = g_n; key = key_n;
      }
    }
    d += two ? 2 : 1;
    if (d < J) {
      if (top_step) { if (blockIdx.x == 0) __syncthreads(); } else grid.sync();
      uint64_t* t = cur; cur = nxt; nxt = t;
    }
    GSNFS_STAMP();
  }
}

__global__ void decode_status_kernel(gsnfs_counts* counts, uint32_t nv, uint32_t occ_bytes, uint32_t status) {
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
  } else if (sum != occ_bytes || level_sizes[0] != 1) {
    status = 1;                                               // header inconsistent with the stream [O12]
  }
  for (int d = 0; d <= depth; ++d)
    if (level_sizes[d] > ctx->max_points) return GSNFS_E_CAPACITY;
  if (occ_bytes + 1 > ctx->occ_cap) return GSNFS_E_CAPACITY;
  if (nv == 0 || status) {                                    // nothing to decode; reported through d_counts
    GSNFS_KERNEL(ctx, st, "decode_status");
    decode_status_kernel<<<1, 1, 0, st>>>(d_counts, status ? 0u : nv, (uint32_t)occ_bytes, status);
    GSNFS_LAUNCH_CHECK(ctx, st);
    return GSNFS_OK;
  }
  DecLevels lv;
  lv.depth = depth;
  uint32_t off = 0;
  for (int d = 0; d <= depth; ++d) {
    lv.size[d] = level_sizes[d];
    lv.off[d] = off;
    if (d < depth) off += level_sizes[d];
  }
  const uint32_t S = (uint32_t)occ_bytes;
  if (S / kScanTile + 2 > ctx->scan_tiles_cap) return GSNFS_E_CAPACITY;
  int per_sm = ctx->occ_cache[7];
  if (per_sm == 0) {
    GSNFS_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, octree_decode_kernel, 256, 0));
    ctx->occ_cache[7] = per_sm;
  }
  if (per_sm < 1) return GSNFS_E_CUDA;
  if (per_sm > 8) per_sm = 8;
  const uint32_t want = (nv + 255) / 256;
  uint32_t grid = (uint32_t)per_sm * (uint32_t)ctx->num_sms;
  if (grid > want) grid = want;
  if (grid < 1) grid = 1;
  unsigned long long* tstamp = ctx->raht_plan->t_dec;
  void* args[] = {(void*)&d_occ, (void*)&S, (void*)&lv, (void*)&ctx->dec_scan, (void*)&ctx->scan_sums,
                  (void*)&ctx->dec_keys_a, (void*)&ctx->dec_keys_b, (void*)&d_voxel_xyz, (void*)&d_voxel_keys, (void*)&d_counts, (void*)&tstamp};
  GSNFS_KERNEL(ctx, st, "octree_decode");
  GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel((void*)octree_decode_kernel, dim3(grid), dim3(256), args, 0, st));
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

}  // namespace gsnfs
