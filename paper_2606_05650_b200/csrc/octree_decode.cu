// Decoder-side position coder (section 2.3, Alg. A.2 / A.3): occupancy bytes -> Morton codes of
// the occupied voxels -> integer coordinates.
//
// The paper expands level by level (count -> prefix-sum -> scatter, 4J launches).  Here the breadth-first
// stream is treated as what it is, a pointer-free tree in level order: with G[n] = sum of popcount(byte m)
// over m < n, the children of stream node n are the nodes G[n] + 1 ... G[n] + popcount(byte n) of the
// breadth-first numbering (root = 0; the leaves continue the numbering after the S internal nodes).  So
//   1. ONE exclusive popcount scan over the whole stream (Alg. A.2 l.10's per-level sums, all at once) ...
//   2. ... whose down-sweep scatters, for every node n and every set bit i of its byte, the word
//      (n << 3 | i) into the child's slot (Alg. A.3 l.4-9: child code = (parent code << 3) + i);
//   3. every node of a middle level, then every leaf, walks up through `parent`, picking up one 3-bit digit per
//      level -- no per-level key lists, no divergence, one coalesced load per hop; neighbouring nodes share
//      ancestors, so the walks hit the same cache lines.
// One cooperative kernel, three grid barriers.
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

constexpr int kDecWalk = 4;           // leaves walked concurrently per thread (memory-level parallelism)

struct DecLevels {
  uint32_t size[GSNFS_MAX_DEPTH + 2];   // |L_d|, d = 0..J
  uint32_t off[GSNFS_MAX_DEPTH + 2];    // stream offset of level d (off[J] = S)
  int depth;
  int mid;                              // level whose codes are materialised between the two walk stages (0 = none)
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
                                                            uint32_t* __restrict__ tile_sums, uint32_t* __restrict__ PD,
                                                            uint64_t* __restrict__ Kmid,
                                                            uint32_t* __restrict__ xyz, uint64_t* __restrict__ keys_out,
                                                            gsnfs_counts* __restrict__ counts, RahtPlan* __restrict__ tl) {
  cg::grid_group grid = cg::this_grid();
  GSNFS_TSTAMP(tl, 0);
  __shared__ uint32_t s_w[9];
  __shared__ uint16_t s_stage[8 * kScanTile];   // a tile's (node-in-tile << 3 | digit) entries on their way out
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int J = lv.depth;
  const uint32_t nv = lv.size[J];
  const uint32_t total_nodes = S + nv;
  if (blockIdx.x == 0 && tid == 0) {
    counts->n_voxels = nv;
    counts->occ_bytes = S;
    counts->status = 0;
    counts->reserved = 0;
  }
  // ---- 1. popcount of every 2048-byte tile of the stream
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
  GSNFS_TSTAMP(tl, 1);
  grid.sync();
  GSNFS_TSTAMP(tl, 2);
  // ---- 2. down-sweep: (parent << 3 | digit) of every child.  The children of a tile are one contiguous id range:
  // staged in shared memory as 16-bit (node-in-tile << 3 | digit), written out coalesced.  The tile's base (number of
  // children before it) is carried from the CTA's previous tile by summing the tile sums in between.
  {
    uint32_t base = 0, prev_t = 0;
    for (uint32_t t = blockIdx.x; t < ntile; t += gridDim.x) {
      {
        uint32_t part = 0;
        for (uint32_t k = prev_t + tid; k < t; k += 256) part += __ldcg(tile_sums + k);
        part = __reduce_add_sync(0xffffffffu, part);
        if (lane == 0) s_w[warp] = part;
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 8; ++k) base += s_w[k];
        __syncthreads();
        prev_t = t;
      }
      const uint32_t i0 = t * kScanTile + tid * 8;
      unsigned long long w = 0ull;                           // bit 8k + i: child i of node i0 + k
      uint32_t nvalid = 0;
      if (i0 + 8 <= S) {
        w = *reinterpret_cast<const unsigned long long*>(occ + i0);
        nvalid = 8;
      } else if (i0 < S) {
        nvalid = S - i0;
        for (uint32_t k = 0; k < nvalid; ++k) w |= (unsigned long long)occ[i0 + k] << (8 * k);
      }
      {   // an internal node without children [O12]: a zero byte among this thread's valid nodes
        unsigned long long z = (w - 0x0101010101010101ull) & ~w & 0x8080808080808080ull;      // bit 8k+7 set iff byte k == 0
        if (nvalid < 8) z &= (1ull << (8 * nvalid)) - 1ull;
        if (z) atomicOr(&counts->status, 1u);
      }
      const uint32_t s = (uint32_t)__popcll(w);
      uint32_t tile_tot;
      uint32_t j = block_excl_scan_256(s, s_w, &tile_tot);                // first child of this thread, tile-local
      const uint32_t ent0 = (uint32_t)tid * 64u;                            // (node-in-tile << 3 | digit) = tid * 64 + bit
      while (w) {
        const uint32_t bit = (uint32_t)__ffsll((long long)w) - 1u;
        w &= w - 1ull;
        s_stage[j++] = (uint16_t)(ent0 + bit);
      }
      __syncthreads();
      const uint32_t tbase = t * kScanTile;
      for (uint32_t q = tid; q < tile_tot; q += 256) {
        const uint32_t idx = base + 1u + q;
        if (idx < total_nodes) {
          const uint32_t e = s_stage[q];
          PD[idx] = ((tbase + (e >> 3)) << 3) | (e & 7u);
        }
      }
      // every node but the root is somebody's child: sum of all popcounts + 1 == number of nodes in the header [O12]
      if (t == ntile - 1 && tid == 0 && base + tile_tot + 1u != total_nodes) atomicOr(&counts->status, 1u);
      base += tile_tot;
      prev_t = t + 1;
      __syncthreads();
    }
  }
  GSNFS_TSTAMP(tl, 3);
  grid.sync();
  GSNFS_TSTAMP(tl, 4);
  // ---- header vs stream, level by level [O12]: with the node count right and no childless node, level e + 1 starts
  // at the header's offset iff its first node is the first child of level e's first node and the node before it is
  // the last child of the node before that
  if (blockIdx.x == 0 && tid >= 1 && tid < J) {
    const uint32_t f = tid + 1 < J ? lv.off[tid + 1] : S;                      // first breadth-first id of level tid + 1
    if ((__ldcg(PD + f) >> 3) != lv.off[tid] || (__ldcg(PD + f - 1u) >> 3) != lv.off[tid] - 1u) atomicOr(&counts->status, 1u);
  }
  // ---- 3. walks.  Stage A: the nodes of a middle level `mid` (chosen on the host) walk up to the root and leave
  // their code in Kmid; stage B: every leaf walks up to its level-`mid` ancestor and prepends that code.
  // kDecWalk walks per thread in flight.  Stale parents (corrupt streams only) are old node ids: always inside P.
  const uint32_t gstride = gridDim.x * 256u;
  const int mid = lv.mid;
  for (int stage = (mid > 0 ? 0 : 1); stage < 2; ++stage) {
    const int hops = stage == 0 ? mid : J - mid;
    const uint32_t cnt = stage == 0 ? lv.size[mid] : nv;
    const uint32_t first = stage == 0 ? lv.off[mid] : S;               // breadth-first id of the level's first node
    for (uint32_t l0 = blockIdx.x * 256u + tid; l0 < cnt; l0 += kDecWalk * gstride) {
      uint32_t id[kDecWalk];
      unsigned long long key[kDecWalk];
#pragma unroll
      for (int u = 0; u < kDecWalk; ++u) { id[u] = first + min(l0 + u * gstride, cnt - 1u); key[u] = 0ull; }
      for (int t = 0; t < hops; ++t) {
        uint32_t pd[kDecWalk];
#pragma unroll
        for (int u = 0; u < kDecWalk; ++u) pd[u] = __ldcg(PD + id[u]);
#pragma unroll
        for (int u = 0; u < kDecWalk; ++u) {
          key[u] |= (unsigned long long)(pd[u] & 7u) << (3 * t);
          id[u] = pd[u] >> 3;
        }
      }
#pragma unroll
      for (int u = 0; u < kDecWalk; ++u) {
        const uint32_t l = l0 + u * gstride;
        if (l < cnt) {
          if (stage == 0) {
            Kmid[l] = key[u];
          } else {
            unsigned long long k = key[u];
            if (mid > 0) {
              const uint32_t a = id[u] - lv.off[mid];                                     // position in level `mid`
              k |= __ldcg(reinterpret_cast<const unsigned long long*>(Kmid) + min(a, lv.size[mid] - 1u)) << (3 * (J - mid));
            }
            emit_leaf(k, l, keys_out, xyz);
          }
        }
      }
    }
    GSNFS_TSTAMP(tl, 5 + 2 * stage);
    if (stage == 0) grid.sync();
    GSNFS_TSTAMP(tl, 6 + 2 * stage);
  }
}

__global__ void decode_status_kernel(gsnfs_counts* counts, uint32_t nv, uint32_t occ_bytes, uint32_t status) {
  counts->n_voxels = nv;
  counts->occ_bytes = occ_bytes;
  counts->status = status;
  counts->reserved = 0;
}

// Header checks that need no device [O12]: the header must describe a tree (one root, no empty level, no level
// larger than the next one: every internal node has >= 1 child) whose internal nodes are the stream's bytes.
bool octree_header_ok(const uint32_t* level_sizes, int depth, uint64_t occ_bytes) {
  if (level_sizes[depth] == 0) return occ_bytes == 0;
  uint64_t sum = 0;
  for (int d = 0; d < depth; ++d) {
    if (level_sizes[d] == 0 || level_sizes[d] > level_sizes[d + 1]) return false;
    sum += level_sizes[d];
  }
  return sum == occ_bytes && level_sizes[0] == 1;
}

int run_octree_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_occ, uint64_t occ_bytes,
                      const uint32_t* level_sizes, int depth, uint32_t* d_voxel_xyz, uint64_t* d_voxel_keys,
                      gsnfs_counts* d_counts) {
  const uint32_t nv = level_sizes[depth];
  const uint32_t status = octree_header_ok(level_sizes, depth, occ_bytes) ? 0u : 1u;
  for (int d = 0; d <= depth; ++d)
    if (level_sizes[d] > ctx->max_points) return GSNFS_E_CAPACITY;
  if (occ_bytes + 1 > ctx->occ_cap || occ_bytes >= (1ull << 29)) return GSNFS_E_CAPACITY;   // parent ids are packed with 3 digit bits
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
  {   // middle level: fewest dependent loads, sum over both stages (0 = one full walk from the leaves)
    lv.mid = 0;
    uint64_t best = (uint64_t)nv * (uint64_t)depth;
    for (int m = 1; m < depth; ++m) {
      const uint64_t cost = (uint64_t)level_sizes[m] * (uint64_t)m + (uint64_t)nv * (uint64_t)(depth - m + 1);
      if (depth >= 6 && cost < best) { best = cost; lv.mid = m; }
    }
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
  const uint32_t want = ((uint32_t)(occ_bytes / 8 > nv ? occ_bytes / 8 : nv) + 255) / 256;
  uint32_t grid = (uint32_t)per_sm * (uint32_t)ctx->num_sms;
  if (grid > want) grid = want;
  if (grid < 1) grid = 1;
  void* args[] = {(void*)&d_occ, (void*)&S, (void*)&lv, (void*)&ctx->scan_sums,
                  (void*)&ctx->dec_parent, (void*)&ctx->dec_kmid, (void*)&d_voxel_xyz, (void*)&d_voxel_keys, (void*)&d_counts,
                  (void*)&ctx->raht_plan};
  GSNFS_KERNEL(ctx, st, "octree_decode");
  GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel((void*)octree_decode_kernel, dim3(grid), dim3(256), args, 0, st));
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

}  // namespace gsnfs
