// Encoder-side position coder: voxelise + Morton (K1/K2), onesweep LSD radix sort (K3), and a fused
// unique + all-levels octree build that emits the breadth-first occupancy stream (K4, K6, K7, K8).
//
// What differs from the paper's design (section 2.2, Alg. A.1): the paper builds L_d level by
// level with J `unique` launches and then runs J OccKernel launches with a binary search per parent.
// Here one pass over the sorted codes does all levels at once.  With h_i = msb(code[i-1] ^ code[i]), sorted
// entry i starts a new node at every depth d >= J - floor(h_i / 3) (and at no depth if it is a duplicate),
// so |L_d|, the index of every node inside its level and each parent's occupancy bits all follow from
// per-level prefix counts of those flags.  The bytes produced are exactly Alg. A.1's.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace gsnfs {

// ------------------------------------------------------------------------------------------------
// K1 + K2: voxelise, Morton-encode, and accumulate the digit histograms of every radix pass.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t spread3(uint32_t v) {   // 21 bits -> every third bit
  uint64_t x = v & 0x1fffffu;
  x = (x | (x << 32)) & 0x001f00000000ffffull;
  x = (x | (x << 16)) & 0x001f0000ff0000ffull;
  x = (x | (x << 8)) & 0x100f00f00f00f00full;
  x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
}

struct VoxParams {
  double lo[3];
  double scale[3];
  double vmax;
};

__device__ __forceinline__ uint32_t voxel_coord(float p, double lo, double scale, double vmax) {
  // [O2]: one rounding for the subtraction, one for the product, no contraction into an FMA.
  const double t = __dsub_rn((double)p, lo);
  const double u = __dmul_rn(t, scale);
  double v = floor(u);
  v = (u < 0.0) ? 0.0 : fmin(v, vmax);      // NaN -> fmin returns vmax: in range, unspecified
  return (uint32_t)v;
}

template <typename KeyT>
__global__ void __launch_bounds__(256) voxelize_kernel(const float* __restrict__ xyz, uint32_t n, VoxParams vp,
                                                       SortPlan plan, KeyT* __restrict__ keys,
                                                       uint32_t* __restrict__ ghist) {
  __shared__ uint32_t s_hist[kSortMaxPasses][256];
  for (int i = threadIdx.x; i < kSortMaxPasses * 256; i += 256) (&s_hist[0][0])[i] = 0;
  __syncthreads();
  const uint32_t stride = gridDim.x * 256u;
  for (uint32_t i0 = blockIdx.x * 256 + threadIdx.x; i0 < n; i0 += 4u * stride) {
    float px[4], py[4], pz[4];                      // four points per thread in flight (the loads are the latency)
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t i = i0 + (uint32_t)u * stride;
      const bool ok = i < n && i >= i0;
      px[u] = ok ? xyz[3 * (size_t)i] : 0.f;
      py[u] = ok ? xyz[3 * (size_t)i + 1] : 0.f;
      pz[u] = ok ? xyz[3 * (size_t)i + 2] : 0.f;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t i = i0 + (uint32_t)u * stride;
      if (i >= n || i < i0) continue;
      const uint32_t vx = voxel_coord(px[u], vp.lo[0], vp.scale[0], vp.vmax);
      const uint32_t vy = voxel_coord(py[u], vp.lo[1], vp.scale[1], vp.vmax);
      const uint32_t vz = voxel_coord(pz[u], vp.lo[2], vp.scale[2], vp.vmax);
      const uint64_t key = spread3(vx) | (spread3(vy) << 1) | (spread3(vz) << 2);
      keys[i] = (KeyT)key;
      for (int p = 0; p < plan.passes; ++p) {
        const uint32_t d = (uint32_t)(key >> plan.shift[p]) & ((1u << plan.bits[p]) - 1u);
        atomicAdd(&s_hist[p][d], 1u);
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < plan.passes * 256; i += 256) {
    const uint32_t c = (&s_hist[0][0])[i];
    if (c) atomicAdd(&ghist[i], c);
  }
}

// ------------------------------------------------------------------------------------------------
// K3: stable LSD radix sort of (code, original index), 8-bit digits, ALL passes in one persistent
// cooperative kernel.  Per pass and tile (4096 keys): warp-level match_any ranking into shared-memory warp
// histograms (onesweep-style), the tile's digit counts are published and added into a per-32-tiles group
// sum, one grid barrier, then every tile gets its global digit offsets from <= 32 + ngroups independent
// loads (no serial look-back chain: at ~1M keys all tiles are co-resident and would all wait on each other),
// shared-memory staged scatter so that global writes are coalesced per digit run, grid barrier, next pass.
// When every CTA owns a single tile the keys, payloads and ranks stay in registers across the barrier.
// ------------------------------------------------------------------------------------------------
constexpr int kSortGroup = 32;     // tiles per histogram group

// Tile = `cnt` consecutive keys starting at `base`; thread (warp, lane) holds items j < ipt at tile-local
// position warp * ipt * 32 + j * 32 + lane (ipt * 256 >= tile stride), so positions grow with (warp, j, lane).
template <typename KeyT>
__device__ __forceinline__ uint32_t sort_load_rank(const KeyT* __restrict__ keys_in, const uint32_t* __restrict__ pay_in,
                                                   uint32_t base, uint32_t cnt, int ipt, int shift, uint32_t mask, bool want_pay,
                                                   KeyT (&key)[kSortItems], uint32_t (&pay)[kSortItems],
                                                   uint32_t (&rank)[kSortItems], uint32_t (*s_whist)[257],
                                                   uint32_t (*s_match)[8][257]) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int i = tid; i < 8 * 257; i += kSortThreads) (&s_whist[0][0])[i] = 0;
  const uint32_t lbase = (uint32_t)(warp * ipt * 32 + lane);
  uint32_t vmask = 0;
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const uint32_t li = lbase + j * 32;
    const bool valid = j < ipt && li < cnt;
    vmask |= (uint32_t)valid << j;
    const uint32_t idx = base + li;
    key[j] = valid ? __ldcg(keys_in + idx) : (KeyT) ~(KeyT)0;
    if (want_pay) pay[j] = valid ? (pay_in ? __ldcg(pay_in + idx) : idx) : 0xffffffffu;
  }
  __syncthreads();
  // lanes holding the same digit: every lane ORs its bit into a per-warp, per-digit mask in shared memory and reads the
  // mask back (bin 256 collects the tail padding); the group's lowest lane clears the mask again.  Two mask sets used
  // alternately, so the clear of item j cannot race with the OR of item j + 1.  ~8 instructions per key where the
  // ballot-per-digit-bit version needed 27 (and the hardware match.any serialises over the distinct values).
  unsigned peers[kSortItems];
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    if (j < ipt) {                                           // warp-uniform
      const bool valid = (vmask >> j) & 1u;
      const uint32_t d = valid ? ((uint32_t)(key[j] >> shift) & mask) : 256u;
      volatile uint32_t* mm = &s_match[j & 1][warp][d];
      atomicOr(const_cast<uint32_t*>(mm), 1u << lane);
      __syncwarp();
      const unsigned m = *mm;
      __syncwarp();
      if ((m & lanemask_lt()) == 0u) *mm = 0u;
      peers[j] = m;
    } else {
      peers[j] = 0xffffffffu;
    }
  }
  __syncwarp();
  // per-warp digit counters: the leader of every peer group adds the group size (shared-memory atomics of
  // one warp execute in program order, so earlier items get the lower ranks) and broadcasts the old value
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    if (j < ipt) {
      const bool valid = (vmask >> j) & 1u;
      const uint32_t d = valid ? ((uint32_t)(key[j] >> shift) & mask) : 256u;
      const unsigned lt = peers[j] & lanemask_lt();
      uint32_t prev = 0;
      if (lt == 0) prev = atomicAdd(&s_whist[warp][d], (uint32_t)__popc(peers[j]));
      prev = __shfl_sync(0xffffffffu, prev, __ffs(peers[j]) - 1);
      rank[j] = prev + __popc(lt);
    }
  }
  __syncthreads();
  return vmask;
}

template <typename KeyT>
__global__ void __launch_bounds__(kSortThreads) sort_coop_kernel(KeyT* ka, KeyT* kb, uint32_t* pa, uint32_t* pb,
                                                                 uint32_t* perm_out, uint32_t n, uint32_t ntiles,
                                                                 uint32_t tstride, int ipt, SortPlan plan,
                                                                 const uint32_t* __restrict__ ghist, uint32_t* tile_hist,
                                                                 uint32_t* group_hist, uint32_t ngroups_cap) {
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) unsigned char s_dyn[];
  KeyT* s_keys = reinterpret_cast<KeyT*>(s_dyn);
  uint32_t* s_pay = reinterpret_cast<uint32_t*>(s_dyn + sizeof(KeyT) * kSortTile);
  __shared__ uint32_t s_whist[8][257];
  __shared__ uint32_t s_match[2][8][257];    // peer masks of the ranking step; all zero between uses (the group leaders clear them)
  __shared__ uint32_t s_dstart[256];
  __shared__ uint32_t s_goff[256];
  __shared__ uint32_t s_scan[9];
  __shared__ uint32_t s_gbase[kSortMaxPasses][256];   // exclusive scan of every pass's global digit histogram

  const int tid = threadIdx.x, warp = tid >> 5;
  for (int i = tid; i < 2 * 8 * 257; i += kSortThreads) (&s_match[0][0][0])[i] = 0;   // (a block barrier precedes the first use)
  const uint32_t ngroups = (ntiles + kSortGroup - 1) / kSortGroup;
  const bool single = ntiles <= gridDim.x;          // one tile per CTA: registers survive the barrier
  KeyT key[kSortItems];
  uint32_t pay[kSortItems];
  uint32_t rank[kSortItems];
  uint32_t vmask = 0;

  {
    uint32_t h[kSortMaxPasses];
#pragma unroll
    for (int p = 0; p < kSortMaxPasses; ++p) h[p] = p < plan.passes ? ghist[p * 256 + tid] : 0u;
#pragma unroll
    for (int p = 0; p < kSortMaxPasses; ++p)
      if (p < plan.passes) s_gbase[p][tid] = block_excl_scan_256(h[p], s_scan, nullptr);
  }
  for (int p = 0; p < plan.passes; ++p) {
    const KeyT* kin = (p & 1) ? kb : ka;
    KeyT* kout = (p & 1) ? ka : kb;
    const uint32_t* pin = (p == 0) ? nullptr : ((p & 1) ? pb : pa);
    uint32_t* pout = (p == plan.passes - 1) ? perm_out : ((p & 1) ? pa : pb);
    const int shift = plan.shift[p];
    const uint32_t mask = (1u << plan.bits[p]) - 1u;
    uint32_t* gh = group_hist + (size_t)(p & 1) * ngroups_cap * 256;
    uint32_t* gh_next = group_hist + (size_t)((p + 1) & 1) * ngroups_cap * 256;

    // ---- phase A: digit counts of every tile -> tile_hist, group sums
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      vmask = sort_load_rank<KeyT>(kin, pin, tile * tstride, min(tstride, n - tile * tstride), ipt, shift, mask, single,
                                   key, pay, rank, s_whist, s_match);
      uint32_t count = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) count += s_whist[w][tid];
      tile_hist[(size_t)tile * 256 + tid] = count;
      if (count) atomicAdd(&gh[(size_t)(tile / kSortGroup) * 256 + tid], count);
      __syncthreads();
    }
    grid.sync();
    // the other parity's group sums are free now: clear them for the next pass
    for (uint32_t i = blockIdx.x * kSortThreads + tid; i < ngroups * 256; i += gridDim.x * kSortThreads) gh_next[i] = 0;

    // ---- phase B: global offsets, scatter
    const uint32_t gbase = s_gbase[p][tid];
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const uint32_t base = tile * tstride;
      const uint32_t cnt = min(tstride, n - base);
      if (!single) vmask = sort_load_rank<KeyT>(kin, pin, base, cnt, ipt, shift, mask, true, key, pay, rank, s_whist, s_match);
      // thread d: exclusive prefix over warps of digit d; tile count of digit d
      uint32_t count = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) {
        const uint32_t c = s_whist[w][tid];
        s_whist[w][tid] = count;
        count += c;
      }
      // digit-d keys in earlier tiles: whole groups from the group sums, the rest of this group tile by tile
      uint32_t excl = 0;
      const uint32_t g = tile / kSortGroup;
      {   // all loads of a batch of 16 are issued before the first use (they are independent L2 hits)
        const uint32_t ntl = tile - g * kSortGroup, tot = g + ntl;
        for (uint32_t i0 = 0; i0 < tot; i0 += 16) {
          uint32_t v[16];
#pragma unroll
          for (int u = 0; u < 16; ++u) {
            const uint32_t i = i0 + u;
            const uint32_t* src = i < g ? gh + (size_t)i * 256 + tid : tile_hist + (size_t)(g * kSortGroup + (i - g)) * 256 + tid;
            v[u] = i < tot ? __ldcg(src) : 0u;
          }
#pragma unroll
          for (int u = 0; u < 16; ++u) excl += v[u];
        }
      }
      const uint32_t dstart = block_excl_scan_256(count, s_scan, nullptr);
      s_dstart[tid] = dstart;
      s_goff[tid] = gbase + excl - dstart;      // global position = s_goff[d] + tile-local sorted position
      __syncthreads();
#pragma unroll
      for (int j = 0; j < kSortItems; ++j) {
        if ((vmask >> j) & 1u) {
          const uint32_t d = (uint32_t)(key[j] >> shift) & mask;
          const uint32_t pos = s_dstart[d] + s_whist[warp][d] + rank[j];
          s_keys[pos] = key[j];
          s_pay[pos] = pay[j];
        }
      }
      __syncthreads();
      for (uint32_t i = tid; i < cnt; i += kSortThreads) {
        const KeyT k = s_keys[i];
        const uint32_t d = (uint32_t)(k >> shift) & mask;
        const uint32_t o = s_goff[d] + i;
        kout[o] = k;
        pout[o] = s_pay[i];
      }
      __syncthreads();
    }
    if (p + 1 < plan.passes) grid.sync();
  }
}

// ------------------------------------------------------------------------------------------------
// K4 + K6 + K7 + K8: unique + all-levels octree build over the sorted codes.
//   t(i) = number of depths at which sorted entry i starts a node:
//          i = 0: J + 1 (depths 0..J); duplicate of i-1: 0; else floor(h_i / 3) + 1 (depths J - floor(h_i/3) .. J).
//   flag_d(i) = t(i) >= J - d + 1.
// ------------------------------------------------------------------------------------------------
template <typename KeyT>
__device__ __forceinline__ int start_levels(const KeyT* __restrict__ keys, uint32_t i, uint32_t n, int J,
                                            uint64_t* key_out) {
  if (i >= n) { *key_out = 0; return 0; }
  const uint64_t k = (uint64_t)keys[i];
  *key_out = k;
  if (i == 0) return J + 1;
  const uint64_t x = k ^ (uint64_t)keys[i - 1];
  if (x == 0) return 0;
  return msb64(x) / 3 + 1;
}

// per-tile counts c_d(tile) for d = 0..J, level-major layout hist[d * ntiles + tile]
template <typename KeyT>
__global__ void __launch_bounds__(256) octree_count_kernel(const KeyT* __restrict__ keys, uint32_t n, int J,
                                                           uint32_t ntiles, uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_cnt[kOctLevels];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < kOctLevels) s_cnt[tid] = 0;
  __syncthreads();
  const uint32_t base = blockIdx.x * (uint32_t)kOctTile + warp * 256;
  uint32_t mine = 0;   // lane d accumulates level d
  for (int it = 0; it < 8; ++it) {
    uint64_t k;
    const int t = start_levels(keys, base + it * 32 + lane, n, J, &k);
    const int tmax = __reduce_max_sync(0xffffffffu, t);          // no lane starts a node above depth J + 1 - tmax
    for (int d = max(0, J + 1 - tmax); d <= J; ++d) {
      const unsigned b = __ballot_sync(0xffffffffu, t >= J - d + 1);
      if (lane == d) mine += __popc(b);
    }
  }
  if (lane <= J) atomicAdd(&s_cnt[lane], mine);
  __syncthreads();
  if (tid <= J) hist[(size_t)tid * ntiles + blockIdx.x] = s_cnt[tid];
}

// one CTA: per level exclusive scan over tiles; level sizes, stream offsets, counts.
__global__ void __launch_bounds__(1024) octree_scan_kernel(const uint32_t* __restrict__ hist,
                                                           uint32_t* __restrict__ tbase, uint32_t ntiles, int J,
                                                           uint32_t n, uint32_t* __restrict__ meta,
                                                           uint32_t* __restrict__ d_level_sizes,
                                                           uint32_t* __restrict__ d_voxel_start,
                                                           gsnfs_counts* __restrict__ d_counts) {
  __shared__ uint32_t s_size[kOctLevels];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int d = warp; d <= J; d += 32) {        // warp per level
    uint32_t carry = 0;
    for (uint32_t b = 0; b < ntiles; b += 32) {
      const uint32_t t = b + lane;
      const uint32_t v = t < ntiles ? hist[(size_t)d * ntiles + t] : 0u;
      uint32_t inc = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t x = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += x;
      }
      if (t < ntiles) tbase[(size_t)d * ntiles + t] = carry + inc - v;
      carry += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) s_size[d] = carry;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t off = 0;
    for (int d = 0; d <= J; ++d) {
      meta[d] = s_size[d];
      meta[kOctLevels + d] = off;       // stream offset of level d (valid for d < J; off[J] = S)
      d_level_sizes[d] = s_size[d];
      if (d < J) off += s_size[d];
    }
    d_counts->n_voxels = s_size[J];
    d_counts->occ_bytes = n ? off : 0u;
    d_counts->status = 0;
    d_counts->reserved = 0;
    d_voxel_start[s_size[J]] = n;
  }
}

template <typename KeyT>
__global__ void __launch_bounds__(256) octree_emit_kernel(const KeyT* __restrict__ keys, uint32_t n, int J,
                                                          uint32_t ntiles, const uint32_t* __restrict__ hist,
                                                          const uint32_t* __restrict__ tbase,
                                                          const uint32_t* __restrict__ meta,
                                                          uint8_t* __restrict__ occ,
                                                          uint64_t* __restrict__ voxel_keys,
                                                          uint32_t* __restrict__ voxel_start) {
  extern __shared__ __align__(16) unsigned char s_dyn[];
  uint32_t* s_stage = reinterpret_cast<uint32_t*>(s_dyn);        // staged occupancy bytes, as words
  __shared__ uint32_t s_wcnt[8][kOctLevels];   // per-warp per-level counts -> exclusive over warps
  __shared__ uint32_t s_cnt[kOctLevels];       // c_d(tile)
  __shared__ uint32_t s_base[kOctLevels];      // nodes of level d started before this tile
  __shared__ uint32_t s_soff[kOctLevels + 1];  // staging offset (bytes) of level e, e < J
  __shared__ uint32_t s_loff[kOctLevels];      // stream offset of level e
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t tile = blockIdx.x;

  if (tid <= J) {
    s_cnt[tid] = hist[(size_t)tid * ntiles + tile];
    s_base[tid] = tbase[(size_t)tid * ntiles + tile];
    s_loff[tid] = meta[kOctLevels + tid];
  }
  __syncthreads();
  if (tid == 0) {
    uint32_t o = 0;
    for (int e = 0; e < J; ++e) { s_soff[e] = o; o += (s_cnt[e] + 1 + 3) & ~3u; }   // word-aligned per level
    s_soff[J] = o;
  }
  __syncthreads();
  const uint32_t stage_words = s_soff[J] >> 2;
  for (uint32_t i = tid; i < stage_words; i += 256) s_stage[i] = 0;

  // pass 1: t values into registers, per-warp per-level counts
  const uint32_t base = tile * (uint32_t)kOctTile + warp * 256;
  int tt[8];
  uint64_t kk[8];
  uint32_t mine = 0;
#pragma unroll
  for (int it = 0; it < 8; ++it) {
    tt[it] = start_levels(keys, base + it * 32 + lane, n, J, &kk[it]);
    const int tmax = __reduce_max_sync(0xffffffffu, tt[it]);
    for (int d = max(0, J + 1 - tmax); d <= J; ++d) {
      const unsigned b = __ballot_sync(0xffffffffu, tt[it] >= J - d + 1);
      if (lane == d) mine += __popc(b);
    }
  }
  if (lane <= J) s_wcnt[warp][lane] = mine;
  __syncthreads();
  if (tid <= J) {                      // exclusive prefix over warps for level tid
    uint32_t run = 0;
    for (int w = 0; w < 8; ++w) { const uint32_t c = s_wcnt[w][tid]; s_wcnt[w][tid] = run; run += c; }
  }
  __syncthreads();

  // pass 2: ranks, voxel list, staged occupancy bits
  uint32_t run = (lane <= J) ? s_wcnt[warp][lane] : 0u;   // lane d: level-d starts in this tile before this warp-iteration
#pragma unroll
  for (int it = 0; it < 8; ++it) {
    const uint32_t i = base + it * 32 + lane;
    const int t = tt[it];
    const uint64_t k = kk[it];
    const int tmax = __reduce_max_sync(0xffffffffu, t);
    const int dmin = max(0, J + 1 - tmax);                       // shallower depths: no lane starts a node
    uint32_t prev_incl = dmin > 0 ? __shfl_sync(0xffffffffu, run, dmin - 1) : 0u;   // tile-local inclusive rank at depth d-1
    for (int d = dmin; d <= J; ++d) {
      const bool f = t >= J - d + 1;
      const unsigned b = __ballot_sync(0xffffffffu, f);
      const uint32_t run_d = __shfl_sync(0xffffffffu, run, d);
      const uint32_t incl = run_d + __popc(b & lanemask_le());
      if (f && d >= 1) {
        // this entry starts a node at depth d; its parent is the prev_incl-th slot of depth d-1
        const uint32_t digit = (uint32_t)(k >> (3 * (J - d))) & 7u;
        const uint32_t sb = s_soff[d - 1] + prev_incl;
        atomicOr(&s_stage[sb >> 2], (1u << digit) << (8 * (sb & 3u)));
      }
      if (f && d == J) {
        const uint32_t v = s_base[J] + incl - 1;
        voxel_keys[v] = k;
        voxel_start[v] = i;
      }
      if (lane == d) run += __popc(b);
      prev_incl = incl;
    }
  }
  __syncthreads();

  // flush: slot s of level e is stream byte loff[e] + base[e] - 1 + s, s = 0..c_e.  Slots 0 and c_e may be
  // shared with neighbouring tiles; any global word holding such a byte (or a byte outside this tile's
  // range of this level) is merged with atomicOr, fully interior words are stored whole.
  uint32_t* occ_w = reinterpret_cast<uint32_t*>(occ);
  for (int e = 0; e < J; ++e) {
    const uint32_t c = s_cnt[e];
    const int64_t g0 = (int64_t)s_loff[e] + (int64_t)s_base[e] - 1;    // stream byte of slot 0 (may be -1 at tile 0)
    const int64_t g1 = g0 + c;
    const int64_t w0 = (g0 < 0 ? 0 : g0) >> 2, w1 = g1 >> 2;
    const uint8_t* sbytes = reinterpret_cast<const uint8_t*>(s_stage) + s_soff[e];
    for (int64_t w = w0 + tid; w <= w1; w += 256) {
      uint32_t val = 0;
      bool interior = true;
#pragma unroll
      for (int bb = 0; bb < 4; ++bb) {
        const int64_t s = (w << 2) + bb - g0;
        if (s >= 0 && s <= (int64_t)c) val |= (uint32_t)sbytes[s] << (8 * bb);
        if (s < 1 || s > (int64_t)c - 1) interior = false;
      }
      if (interior) occ_w[w] = val;
      else if (val) atomicOr(&occ_w[w], val);
    }
  }
}

// ------------------------------------------------------------------------------------------------
static SortPlan make_sort_plan(int depth) {
  SortPlan p{};
  const int total = 3 * depth;
  p.passes = (total + 7) / 8;
  int shift = 0;
  for (int i = 0; i < p.passes; ++i) {           // spread the bits evenly over the passes
    const int b = (total - shift + (p.passes - i) - 1) / (p.passes - i);
    p.shift[i] = shift;
    p.bits[i] = b;
    shift += b;
  }
  return p;
}

template <typename KeyT>
static int encode_impl(gsnfs_ctx* ctx, cudaStream_t st, const float* d_xyz, uint32_t n, const VoxParams& vp,
                       int depth, uint8_t* d_occ, uint64_t occ_capacity, uint32_t* d_level_sizes, uint32_t* d_perm,
                       uint64_t* d_voxel_keys, uint32_t* d_voxel_start, gsnfs_counts* d_counts) {
  const SortPlan plan = make_sort_plan(depth);
  KeyT* ka = reinterpret_cast<KeyT*>(ctx->keys_a);
  KeyT* kb = reinterpret_cast<KeyT*>(ctx->keys_b);

  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(ctx->hist, 0, ctx->sort_zero_bytes, st));
  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(d_occ, 0, occ_capacity, st));
  if (n) {
    const uint32_t vwant = (n + 1023u) / 1024u, vcap = (uint32_t)ctx->num_sms * 8u;
    const int vgrid = (int)(vwant < vcap ? vwant : vcap);
    GSNFS_KERNEL(ctx, st, "voxelize_morton_hist");
    voxelize_kernel<KeyT><<<vgrid, 256, 0, st>>>(d_xyz, n, vp, plan, ka, ctx->hist);
    GSNFS_LAUNCH_CHECK(ctx, st);
    const size_t smem = (sizeof(KeyT) + 4) * (size_t)kSortTile;
    {
      const int slot = sizeof(KeyT) == 8 ? 5 : 6;
      int per_sm = ctx->occ_cache[slot];
      if (per_sm == 0) {
        GSNFS_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sort_coop_kernel<KeyT>, kSortThreads, smem));
        ctx->occ_cache[slot] = per_sm;
      }
      if (per_sm < 1) { snprintf(ctx->err, sizeof(ctx->err), "sort kernel does not fit on an SM"); return GSNFS_E_CUDA; }
      // balanced tiling: the tile count is (close to) a multiple of the co-resident grid, so that every SM
      // ranks and scatters the same number of keys in every pass; tile stride <= kSortTile, a multiple of 32
      const uint32_t cap = (uint32_t)per_sm * (uint32_t)ctx->num_sms;
      const uint32_t rounds = (n + cap * (uint32_t)kSortTile - 1u) / (cap * (uint32_t)kSortTile);
      uint32_t tstride = ((n + cap * rounds - 1u) / (cap * rounds) + 31u) & ~31u;
      if (tstride < 1024u) tstride = 1024u;
      const uint32_t stiles = (n + tstride - 1u) / tstride;
      int ipt = (int)((tstride + kSortThreads - 1u) / kSortThreads);
      uint32_t grid = cap < stiles ? cap : stiles;
      KeyT* kbuf_a = ka;
      KeyT* kbuf_b = kb;
      uint32_t* pbuf_a = ctx->pay_a;
      uint32_t* pbuf_b = ctx->pay_b;
      uint32_t nn = n;
      SortPlan pl = plan;
      const uint32_t* gh = ctx->hist;
      uint32_t* th = ctx->sort_tile_hist;
      uint32_t* grp = ctx->sort_group_hist;
      uint32_t gcap = ctx->sort_groups_cap;
      uint32_t ntl = stiles;
      void* args[] = {(void*)&kbuf_a, (void*)&kbuf_b, (void*)&pbuf_a, (void*)&pbuf_b, (void*)&d_perm, (void*)&nn, (void*)&ntl,
                      (void*)&tstride, (void*)&ipt, (void*)&pl,
                      (void*)&gh, (void*)&th, (void*)&grp, (void*)&gcap};
      GSNFS_KERNEL(ctx, st, "radix_sort");
      GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel((void*)sort_coop_kernel<KeyT>, dim3(grid), dim3(kSortThreads), args, smem, st));
      GSNFS_LAUNCH_CHECK(ctx, st);
    }
    const KeyT* sorted = (plan.passes & 1) ? kb : ka;
    const uint32_t otiles = (n + kOctTile - 1) / kOctTile;
    GSNFS_KERNEL(ctx, st, "octree_count");
    octree_count_kernel<KeyT><<<otiles, 256, 0, st>>>(sorted, n, depth, otiles, ctx->oct_hist);
    GSNFS_LAUNCH_CHECK(ctx, st);
    GSNFS_KERNEL(ctx, st, "octree_scan");
    octree_scan_kernel<<<1, 1024, 0, st>>>(ctx->oct_hist, ctx->oct_base, otiles, depth, n, ctx->oct_meta,
                                           d_level_sizes, d_voxel_start, d_counts);
    GSNFS_LAUNCH_CHECK(ctx, st);
    const size_t esmem = (size_t)depth * (kOctTile + 4);
    GSNFS_KERNEL(ctx, st, "octree_emit");
    octree_emit_kernel<KeyT><<<otiles, 256, esmem, st>>>(sorted, n, depth, otiles, ctx->oct_hist, ctx->oct_base,
                                                         ctx->oct_meta, d_occ, d_voxel_keys, d_voxel_start);
    GSNFS_LAUNCH_CHECK(ctx, st);
  } else {
    GSNFS_CUDA_OK(ctx, cudaMemsetAsync(d_level_sizes, 0, sizeof(uint32_t) * (depth + 1), st));
    GSNFS_CUDA_OK(ctx, cudaMemsetAsync(d_counts, 0, sizeof(gsnfs_counts), st));
    GSNFS_CUDA_OK(ctx, cudaMemsetAsync(d_voxel_start, 0, sizeof(uint32_t), st));
  }
  return GSNFS_OK;
}

int octree_encode_setup(gsnfs_ctx* ctx) {
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(sort_coop_kernel<uint64_t>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)((8 + 4) * kSortTile)));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(sort_coop_kernel<uint32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)((4 + 4) * kSortTile)));
  const int esmem = GSNFS_MAX_DEPTH * (kOctTile + 4);
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(octree_emit_kernel<uint64_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, esmem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(octree_emit_kernel<uint32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, esmem));
  return GSNFS_OK;
}

int run_octree_encode(gsnfs_ctx* ctx, cudaStream_t st, const float* d_xyz, uint32_t n, const double lo[3],
                      const double scale[3], int depth, uint8_t* d_occ, uint64_t occ_capacity,
                      uint32_t* d_level_sizes, uint32_t* d_perm, uint64_t* d_voxel_keys, uint32_t* d_voxel_start,
                      gsnfs_counts* d_counts) {
  VoxParams vp;
  for (int a = 0; a < 3; ++a) { vp.lo[a] = lo[a]; vp.scale[a] = scale[a]; }
  vp.vmax = (double)((1u << depth) - 1u);
  if (3 * depth <= 32)
    return encode_impl<uint32_t>(ctx, st, d_xyz, n, vp, depth, d_occ, occ_capacity, d_level_sizes, d_perm,
                                 d_voxel_keys, d_voxel_start, d_counts);
  return encode_impl<uint64_t>(ctx, st, d_xyz, n, vp, depth, d_occ, occ_capacity, d_level_sizes, d_perm,
                               d_voxel_keys, d_voxel_start, d_counts);
}

}  // namespace gsnfs
