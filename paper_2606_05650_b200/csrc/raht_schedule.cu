// RAHT schedule ("prelude", section 3.2-3.3, Alg. A.4 / A.5): which entries of the Morton-sorted voxel list
// are siblings at which binary level, with which weights -- computed from the codes alone, shared by the forward and
// the inverse transform.
//
// The paper builds 3J active lists with 3J flag kernels and 3J masked_select compactions.  Here the sorted list is cut
// into tiles of 256 entries; with g_k = msb(code[k-1] xor code[k]) the "height" of the boundary in front of entry k,
// the binary tree of Alg. A.4 is the Cartesian tree of the heights: entry k > 0 is the right sibling of the butterfly
// at level g_k + 1 (A.4 l.10's flag test), its left node spans [l, k) and its right node [k, r), l / r being the nearest
// boundaries to the left / right with a GREATER height, and the weights W0, W1 are the leaf-weight sums of the two
// spans (A.4 l.8 run lengths).  A butterfly is LOCAL to a tile when both bounds lie inside it (or at a tile edge whose
// outer boundary is higher).  The entries that are not local (at most 2 * 3J + 1 per tile: the strict prefix / suffix
// maxima of the heights; 3.7 % at the headline config) become the nodes of the next PHASE,
// which is processed the same way, until one node -- the DC -- is left.
//
// One CTA per tile, one thread per entry: the tile's boundaries are binned into per-height 256-bit masks in shared
// memory, a suffix OR over the heights (one warp per mask word) turns them into ">= height" masks, and l / r are two
// bit scans.  Local butterflies are ordered by their DEPTH in the tile's forest
// (number of local ancestors: +1 on the boundaries strictly inside every local butterfly's span, then a prefix sum),
// deepest first: butterflies of equal depth are independent, so the transform kernels need one barrier per depth
// (~10 per tile, the minimum) instead of one per non-empty binary level (30-40 in the upper phases).  a =
// sqrt(W0/(W0+W1)), b = sqrt(W1/(W0+W1)) in fp32 with IEEE division and square root.  All phases run in one cooperative
// launch, one grid barrier per phase; pending lists are never compacted (the next phase maps entry -> (source tile,
// rank) through per-256-tile bucket sums).
#include <cooperative_groups.h>
#include <cstddef>

#include "merge_long.cuh"
#include "raht.cuh"

namespace cg = cooperative_groups;

namespace gsnfs {

namespace {

constexpr int T = kRahtTile;

__device__ __forceinline__ PendRec ld_pend(const PendRec* p) {
  const uint4 v = __ldcg(reinterpret_cast<const uint4*>(p));
  PendRec r; r.klo = v.x; r.khi = v.y; r.vidx = v.z; r.w = v.w;
  return r;
}
__device__ __forceinline__ uint64_t pend_key(const PendRec& r) { return (uint64_t)r.klo | ((uint64_t)r.khi << 32); }

// Block-wide search in the exclusive prefix E of vals[0..n) (all vals > 0 where it matters): returns the
// index i and E(i) with E(i) <= target < E(i+1).  All 256 threads must call it.
struct PrefixHit { uint32_t idx, before; };
__device__ PrefixHit block_prefix_find(const uint32_t* vals, uint32_t n, uint32_t target, uint32_t* s_scan /*9*/,
                                       uint32_t* s_hit /*2*/) {
  uint32_t running = 0;
  if (threadIdx.x == 0) { s_hit[0] = 0; s_hit[1] = 0; }
  __syncthreads();
  for (uint32_t base = 0; base < n; base += 256) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t v = i < n ? __ldcg(vals + i) : 0u;
    uint32_t tot;
    const uint32_t ex = block_excl_scan_256(v, s_scan, &tot) + running;
    if (v && ex <= target && target < ex + v) { s_hit[0] = i; s_hit[1] = ex; }
    running += tot;
  }
  __syncthreads();
  PrefixHit h;
  h.idx = s_hit[0]; h.before = s_hit[1];
  __syncthreads();
  return h;
}

// Packed 64-bit exclusive scan over a 256-thread block (two barriers).
__device__ __forceinline__ uint64_t block_excl_scan_256_u64(uint64_t v, uint64_t* s_warp /*>= 9*/, uint64_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint64_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) s_warp[warp] = inc;
  __syncthreads();
  uint64_t before = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) { const uint64_t x = s_warp[w]; if (w < warp) before += x; tot += x; }
  *total = tot;
  return inc - v + before;           // s_warp may be rewritten only after the caller's next barrier
}

struct __align__(16) TileSmem {   // double buffered: tile i+1 fills its set while stragglers still read tile i's
  uint64_t key[T];
  uint32_t ge[65][8];        // [h][word]: tile boundaries of height >= h ([64] stays empty); rows are read as 2 x uint4
  uint32_t wpre[T + 1];      // tile-local exclusive prefix of the entry weights
  int diff[T + 1];           // +1 / -1 marks of the local butterflies' spans
  uint32_t hist[64];         // butterflies per depth bucket
  uint32_t start[64];
  uint32_t pmask[8];
  uint32_t nonunit[8];       // per warp: some entry weight != 1 (phase 1: the transform kernels scale those rows [R2])
  uint64_t edge[2];
  uint64_t scan64[9];
  int dmax;
  int pad[3];
};
static_assert(sizeof(TileSmem) % 16 == 0 && offsetof(TileSmem, ge) % 16 == 0, "TileSmem::ge rows are read as uint4");

__global__ void __launch_bounds__(256) raht_schedule_kernel(
    const uint64_t* __restrict__ keys, const uint32_t* __restrict__ weights, uint32_t n_host,
    gsnfs_counts* __restrict__ counts, SchedPools sp, RahtPlan* __restrict__ plan, uint32_t* __restrict__ sticky) {
  cg::grid_group grid = cg::this_grid();
  __shared__ __align__(16) TileSmem s_tile[2];
  __shared__ uint32_t s_E[2 * T + 1];      // exclusive prefix of source-tile pending counts
  __shared__ uint32_t s_scan[9];
  __shared__ uint32_t s_hit[2];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // a frame the decoder flagged corrupt (status != 0) has no transform: N_v = 0 makes every later kernel a no-op
  const uint32_t Nv = counts ? (counts->status ? 0u : min(counts->n_voxels, n_host)) : n_host;
  uint32_t M = Nv, toff = 0, boff = 0;
  uint32_t toff_prev = 0, boff_prev = 0, ntiles_prev = 0, poff = 0;
  bool overflow = false;
  int p = 1;
  int cur = 0;
  if (blockIdx.x == 0 && tid == 0) {
    plan->M[0] = 0; plan->M[1] = Nv; plan->poff[1] = 0; plan->toff[1] = 0; plan->nphases = 1;   // overflow / invalid: cleared by the host
  }
  for (int i = tid; i < (int)(sizeof(s_tile) / 4); i += 256) reinterpret_cast<uint32_t*>(s_tile)[i] = 0u;
  __syncthreads();
  GSNFS_TSTAMP(plan, 0);
  while (true) {
    const uint32_t ntiles = (M + T - 1) / T;
    const uint32_t nb = (ntiles + 255) / 256;
    const uint32_t nb_prev = (ntiles_prev + 255) / 256;
    if (toff + ntiles > sp.hdr_cap || boff + nb > sp.bsum_cap) {      // uniform over the grid
      overflow = true;
      break;
    }
    // phase 1: the global inputs of a tile (code, leaf weight or run bounds, edge codes) are loaded one tile ahead, so
    // that their latency overlaps the previous tile's work
    uint64_t pf_key = ~0ull, pf_edge = 0ull;
    uint32_t pf_a = 0, pf_b = 0;
    auto preload = [&](uint32_t tile) {
      if (tile >= ntiles) return;
      const uint32_t ks = tile * T;
      const uint32_t cnt = min((uint32_t)T, M - ks);
      if ((uint32_t)tid < cnt) {
        const uint32_t v = ks + tid;
        pf_key = keys[v];
        if (sp.perm) { pf_a = sp.vstart[v]; pf_b = sp.vstart[v + 1]; }
        else pf_a = weights ? weights[v] : 1u;
      }
      if (tid == 0 && ks > 0) pf_edge = keys[ks - 1];
      if (tid == 32 && ks + cnt < M) pf_edge = keys[ks + cnt];
    };
    if (p == 1) preload(blockIdx.x);
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      TileSmem& S = s_tile[cur];
      cur ^= 1;
      const uint32_t ks = tile * T;
      const uint32_t cnt = min((uint32_t)T, M - ks);
      const bool valid = (uint32_t)tid < cnt;
      const bool has_prev = ks > 0, has_next = ks + cnt < M;
      uint32_t vidx = 0xffffffffu, went = 0;
      uint64_t mk = ~0ull;
      if (p == 1) {
        if (valid) {
          vidx = ks + tid;
          mk = pf_key;
          if (sp.perm) {
            went = pf_b - pf_a;
            if (went >= kLongRun) plan->has_long = 1u;        // the forward kernel runs the chunk pre-pass first
            sp.gsrc[vidx] = sp.perm[pf_a];
            sp.weights_out[vidx] = went;
          } else {
            went = pf_a;
          }
        }
        if (tid == 0) S.edge[0] = has_prev ? pf_edge : 0ull;
        if (tid == 32) S.edge[1] = has_next ? pf_edge : 0ull;
        preload(tile + gridDim.x);
      } else {
        // entry g of this phase = pending entry (g - E(t)) of the previous phase's tile t, E(t) <= g < E(t+1).  Every
        // tile has >= 1 pending entry (its first), so the 256 entries of this tile and their two neighbours lie in
        // the 512 source tiles that start at the 256-tile block holding entry ks.
        const PrefixHit hb = block_prefix_find(sp.bsum + boff_prev, nb_prev, ks, s_scan, s_hit);
        const uint32_t tb = hb.idx * 256;
        {
          const uint32_t t0 = tb + 2 * tid, t1 = t0 + 1;
          const uint32_t v0 = t0 < ntiles_prev ? __ldcg(sp.tile_pend + toff_prev + t0) : 0u;
          const uint32_t v1 = t1 < ntiles_prev ? __ldcg(sp.tile_pend + toff_prev + t1) : 0u;
          uint32_t tot;
          const uint32_t ex = block_excl_scan_256(v0 + v1, s_scan, &tot);
          s_E[2 * tid] = hb.before + ex;
          s_E[2 * tid + 1] = hb.before + ex + v0;
          if (tid == 0) s_E[2 * T] = hb.before + tot;
        }
        __syncthreads();
        auto fetch = [&](uint32_t g) -> PendRec {
          if (g < s_E[0]) {            // only for g = ks - 1: the last pending entry of the tile before the window
            const uint32_t c = __ldcg(sp.tile_pend + toff_prev + tb - 1);
            return ld_pend(sp.pend + (size_t)(toff_prev + tb - 1) * kPendCap + min(c - 1u, (uint32_t)kPendCap - 1u));
          }
          uint32_t lo = 0, hi = 2 * T - 1;               // last i in [0, 2T) with s_E[i] <= g
          while (lo < hi) { const uint32_t mid = (lo + hi + 1) >> 1; if (s_E[mid] <= g) lo = mid; else hi = mid - 1; }
          const uint32_t rank = min(g - s_E[lo], (uint32_t)kPendCap - 1u);
          return ld_pend(sp.pend + (size_t)(toff_prev + min(tb + lo, ntiles_prev - 1u)) * kPendCap + rank);
        };
        if (valid) {
          const PendRec pr = fetch(ks + tid);
          vidx = pr.vidx; went = pr.w;
          mk = pend_key(pr);
        }
        if (tid == 32 && has_prev) S.edge[0] = pend_key(fetch(ks - 1));
        if (tid == 64 && has_next) S.edge[1] = pend_key(fetch(ks + cnt));
      }
      S.key[tid] = mk;
      __syncthreads();                                                                       // (1)
      // heights of the tile's boundaries; the codes must be sorted and unique (gsnfs.h): a violation is reported
      int h = 64;
      if (valid) {
        const uint64_t left = tid > 0 ? S.key[tid - 1] : S.edge[0];
        if (((tid > 0 || has_prev) && left >= mk) || went == 0u) plan->invalid = 1u;       // (weight 0: no transform [R1])
        if (tid > 0) {
          const uint64_t x = left ^ mk;
          h = x ? msb64(x) : 0;
          atomicOr(&S.ge[h][warp], 1u << lane);
        }
      }
      const uint64_t x_first = S.edge[0] ^ S.key[0];
      const uint64_t x_end = S.edge[1] ^ S.key[cnt - 1];
      const int hfirst = has_prev ? (x_first ? msb64(x_first) : 0) : 64;
      const int hend = has_next ? (x_end ? msb64(x_end) : 0) : 64;
      __syncthreads();                                                                       // (2)
      {   // ">= height" masks: suffix OR over the 64 heights, warp w owns mask word w
        uint32_t lo = S.ge[lane][warp], hi = S.ge[32 + lane][warp];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const uint32_t a = __shfl_down_sync(0xffffffffu, lo, o), b = __shfl_down_sync(0xffffffffu, hi, o);
          if (lane + o < 32) { lo |= a; hi |= b; }
        }
        lo |= __shfl_sync(0xffffffffu, hi, 0);
        S.ge[lane][warp] = lo;
        S.ge[32 + lane][warp] = hi;
      }
      __syncthreads();                                                                       // (3)
      bool local = false;
      uint32_t l = 0, r = cnt;
      if (valid && tid > 0) {
        const uint4* G4 = reinterpret_cast<const uint4*>(S.ge[h + 1]);
        const uint4 ga = G4[0], gb = G4[1];
        const uint32_t G[8] = {ga.x, ga.y, ga.z, ga.w, gb.x, gb.y, gb.z, gb.w};
        bool lf = false, rf = false;
#pragma unroll
        for (int w = 7; w >= 0; --w) {          // highest set bit below this entry
          uint32_t m = G[w];
          if (w == warp) m &= lanemask_lt();
          if (w <= warp && !lf && m) { l = (uint32_t)(w * 32 + 31 - __clz(m)); lf = true; }
        }
#pragma unroll
        for (int w = 0; w < 8; ++w) {           // lowest set bit above it
          uint32_t m = G[w];
          if (w == warp) m &= ~lanemask_le();
          if (w >= warp && !rf && m) { r = (uint32_t)(w * 32 + __ffs(m) - 1); rf = true; }
        }
        if (!lf) { l = 0; lf = hfirst > h; }
        if (!rf) { r = cnt; rf = hend > h; }
        local = lf && rf;
        if (local) { atomicAdd(&S.diff[l + 1], 1); atomicAdd(&S.diff[r], -1); }
      }
      __syncthreads();                                                                       // (4)
      // one packed scan: weights (exclusive prefix, low 40 bits) and span marks (inclusive prefix = 1 + number of
      // local ancestors, high 24 bits, two's complement)
      int depth = 0;
      {
        const uint64_t v = (uint64_t)went + ((uint64_t)(int64_t)S.diff[tid] << 40);
        uint64_t tot;
        const uint64_t ex = block_excl_scan_256_u64(v, S.scan64, &tot);                      // (5) inside
        S.wpre[tid] = (uint32_t)(ex & 0xffffffffffull);
        if (tid == 0) S.wpre[T] = (uint32_t)(tot & 0xffffffffffull);
        depth = (int)((int64_t)(ex + v) >> 40) - 1;
      }
      {
        const int dm = __reduce_max_sync(0xffffffffu, local ? depth : -1);
        if (lane == 0 && dm >= 0) atomicMax(&S.dmax, dm + 1);
      }
      const unsigned pend_b = __ballot_sync(0xffffffffu, valid && !local);
      const unsigned nu_b = __ballot_sync(0xffffffffu, valid && went != 1u);
      if (lane == 0) { S.pmask[warp] = pend_b; S.nonunit[warp] = nu_b; }
      __syncthreads();                                                                       // (6)
      const int dmax = S.dmax - 1;                       // stored biased by one: 0 = no butterfly in the tile
      float fa = 0.f, fb = 0.f;
      uint32_t bucket = 0, brank = 0;                    // deepest butterflies first: bucket 0 = depth dmax
      if (local) {
        bucket = (uint32_t)min(max(dmax - depth, 0), 63);
        const uint32_t pk = S.wpre[tid];
        const uint32_t W0 = pk - S.wpre[l], W1 = S.wpre[r] - pk;          // entries >= cnt carry weight 0: wpre[cnt] = total
        const float w0 = (float)W0, w1 = (float)W1, ws = (float)(W0 + W1);
        fa = __fsqrt_rn(__fdiv_rn(w0, ws));
        fb = __fsqrt_rn(__fdiv_rn(w1, ws));
        // rank inside the bucket: one shared-memory atomic per group of equal buckets in the warp (the order inside a
        // bucket is free: its butterflies are independent)
        const unsigned peers = __match_any_sync(__activemask(), bucket);
        const int leader = __ffs(peers) - 1;
        uint32_t base = 0;
        if (lane == leader) base = atomicAdd(&S.hist[bucket], (uint32_t)__popc(peers));
        brank = __shfl_sync(peers, base, leader) + __popc(peers & lanemask_lt());
      }
      __syncthreads();                                                                       // (7)
      const uint32_t nseg = (uint32_t)min(dmax + 1, 64);
      if (warp == 0) {                      // exclusive scan of the bucket counts (depths 0..dmax are all non-empty)
        const uint32_t t0 = S.hist[2 * lane], t1 = S.hist[2 * lane + 1];
        uint32_t inc = t0 + t1;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
        const uint32_t ex = inc - (t0 + t1);
        S.start[2 * lane] = ex;
        S.start[2 * lane + 1] = ex + t0;
        RahtTileHdr* h_out = sp.hdr + toff + tile;
        const uint32_t le0 = 2u * lane < nseg ? ex + t0 : 0u, le1 = 2u * lane + 1u < nseg ? ex + t0 + t1 : 0u;
        reinterpret_cast<uint32_t*>(h_out->lev_end)[lane] = le0 | (le1 << 16);
      }
      __syncthreads();                                                                       // (8)
      const size_t tbase = (size_t)(toff + tile) * T;
      RahtTileHdr* h_out = sp.hdr + toff + tile;
      if (local) {
        uint4 rr;
        rr.x = (uint32_t)tid | (l << 8) | (bucket << 16);
        rr.y = __float_as_uint(fa);
        rr.z = __float_as_uint(fb);
        rr.w = vidx;
        sp.rec[tbase + min(S.start[bucket] + brank, (uint32_t)T - 1u)] = rr;
      }
      uint32_t np = 0, before = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) { const uint32_t c = __popc(S.pmask[w]); if (w < warp) before += c; np += c; }
      if (valid && !local) {
        // pending node = this entry plus everything merged into it: up to the next pending entry
        const uint32_t rank = before + __popc(S.pmask[warp] & lanemask_lt());
        uint32_t nxt = cnt;                                          // next pending entry after tid
        {
          unsigned m = S.pmask[warp] & ~lanemask_le();
          int w = warp;
          while (m == 0 && ++w < 8) m = S.pmask[w];
          if (m) nxt = (uint32_t)(w * 32 + __ffs(m) - 1);
        }
        if (rank < (uint32_t)kPendCap) {                             // always, for sorted unique codes
          uint4 pr;
          pr.x = (uint32_t)mk; pr.y = (uint32_t)(mk >> 32); pr.z = vidx; pr.w = S.wpre[nxt] - S.wpre[tid];
          reinterpret_cast<uint4*>(sp.pend)[(size_t)(toff + tile) * kPendCap + rank] = pr;
        }
      }
      if (tid < 8) h_out->pendmask[tid] = S.pmask[tid];
      if (tid == 0) {
        if (np > (uint32_t)kPendCap) plan->invalid = 1u;             // impossible for sorted unique codes
        h_out->npend = np;
        uint32_t nu = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) nu |= S.nonunit[w];
        h_out->nent = cnt | (nseg << 16) | (nu ? 0x80000000u : 0u);
        h_out->nmerge = cnt - np;
        h_out->pend_off = 0;
        sp.tile_pend[toff + tile] = np;
        atomicAdd(&sp.bsum[boff + tile / 256], np);
      }
      __syncthreads();                                                                       // (9) all reads of this set done
      // reset this tile's set for its next use (two tiles from now): ordered before that use by the barriers of the
      // tile in between
      S.diff[tid] = 0;
      if (tid == 0) { S.diff[T] = 0; S.dmax = 0; }
      for (int i = tid; i < 65 * 8; i += 256) (&S.ge[0][0])[i] = 0;
      if (tid < 64) S.hist[tid] = 0;
    }
    // side job (p >= 2), after the CTA's own tiles: exclusive offsets of the previous phase's pending lists -> its
    // tile headers (the pending-row pool positions the transform kernels use).  Taken from the END of the grid: the few
    // tiles of a small phase sit at its beginning.
    if (p >= 2) {
      for (uint32_t b = gridDim.x - 1u - blockIdx.x; b < nb_prev; b += gridDim.x) {
        uint32_t part = 0;
        for (uint32_t i = tid; i < b; i += 256) part += __ldcg(sp.bsum + boff_prev + i);
        part = __reduce_add_sync(0xffffffffu, part);
        if (lane == 0) s_scan[warp] = part;
        __syncthreads();
        uint32_t bpre = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) bpre += s_scan[w];
        __syncthreads();
        const uint32_t t = b * 256 + tid;
        const uint32_t v = t < ntiles_prev ? __ldcg(sp.tile_pend + toff_prev + t) : 0u;
        const uint32_t ex = block_excl_scan_256(v, s_scan, nullptr);
        if (t < ntiles_prev) sp.hdr[toff_prev + t].pend_off = bpre + ex;
      }
    }
    GSNFS_TSTAMP(plan, 2 * p - 1);
    grid.sync();
    GSNFS_TSTAMP(plan, 2 * p);
    uint32_t part = 0;
    for (uint32_t i = tid; i < nb; i += 256) part += __ldcg(sp.bsum + boff + i);
    part = __reduce_add_sync(0xffffffffu, part);
    if (lane == 0) s_scan[warp] = part;
    __syncthreads();
    uint32_t M_next = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) M_next += s_scan[w];
    __syncthreads();
    const uint32_t poff_next = (p == 1) ? 0u : poff + M;
    if (blockIdx.x == 0 && tid == 0) {
      plan->M[p + 1] = M_next; plan->poff[p + 1] = poff_next; plan->toff[p + 1] = toff + ntiles;
    }
    // no progress (M_next >= M) happens only for codes that are not sorted and unique: stop instead of looping
    if ((uint64_t)poff_next + M_next > sp.pool_rows || (M_next > 1 && (p + 1 > kRahtMaxPhases || M_next >= M))) {
      overflow = true;
      break;
    }
    if (M_next <= 1) break;
    toff_prev = toff; boff_prev = boff; ntiles_prev = ntiles;
    poff = poff_next;
    toff += ntiles; boff += nb;
    M = M_next;
    ++p;
  }
  if (blockIdx.x == 0 && tid == 0) {
    plan->nphases = (uint32_t)p;
    if (overflow || *(volatile uint32_t*)&plan->invalid) {   // loud: the transform kernels write nothing; the caller sees status bit 1
      plan->overflow = 1;
      if (counts) atomicOr(&counts->status, 2u);
      *sticky = 1u;
      __threadfence_system();
    }
  }
}

}  // namespace

int launch_raht_schedule(gsnfs_ctx* ctx, cudaStream_t st, const uint64_t* d_keys, const uint32_t* d_weights,
                         uint32_t n_voxels, gsnfs_counts* d_counts, const SchedPools& sp_in) {
  SchedPools sp = sp_in;
  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(ctx->raht_bsum, 0, sizeof(uint32_t) * ctx->raht_bsum_cap, st));
  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(&ctx->raht_plan->overflow, 0, 3 * sizeof(uint32_t), st));   // overflow, invalid, has_long
  int per_sm = ctx->occ_cache[0];
  if (per_sm == 0) {
    GSNFS_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, raht_schedule_kernel, 256, 0));
    ctx->occ_cache[0] = per_sm;
  }
  if (per_sm < 1) { snprintf(ctx->err, sizeof(ctx->err), "raht schedule kernel does not fit on an SM"); return GSNFS_E_CUDA; }
  const uint32_t want = (n_voxels + T - 1) / T;
  const uint32_t cap = (uint32_t)per_sm * (uint32_t)ctx->num_sms;
  const int grid = (int)max(1u, min(cap, want));
  void* args[] = {(void*)&d_keys, (void*)&d_weights, (void*)&n_voxels, (void*)&d_counts, (void*)&sp, (void*)&ctx->raht_plan,
                  (void*)&ctx->d_flags};
  GSNFS_KERNEL(ctx, st, "raht_schedule");
  GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel((void*)raht_schedule_kernel, dim3(grid), dim3(256), args, 0, st));
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

}  // namespace gsnfs
