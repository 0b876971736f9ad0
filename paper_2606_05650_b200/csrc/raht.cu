// Region-Adaptive Hierarchical Transform, forward (+ dead-zone quantiser) and inverse
// (section 3, Eq. (1), Appendix D, Alg. A.4-A.6).
//
// What is computed is exactly Alg. A.6: N_v - 1 butterflies, each at the binary level l = h + 1 where
// h = msb(M[i-1] xor M[i]) is the highest bit in which the right sibling's first voxel differs from its
// predecessor (equivalent to the flag test of A.4 l.10), with run-length weights W_l (A.4 l.8).
//
// What differs from the paper's design: the paper launches one kernel per binary level (3J launches over
// a global active list that is re-compacted 3J times).  Here the sorted voxel list is cut into tiles of
// kRahtTile entries whose rows are staged in shared memory; every butterfly whose two sibling sub-trees
// lie inside one tile is done there, level by level, with __syncthreads() between levels.  What is left
// of a tile is a short list of still-pending low-pass nodes (at most 2*3J+1, a few per cent in practice);
// those lists are concatenated and the same tile procedure is repeated on them ("phase" 2, 3, ...) until
// one node -- the DC -- remains.  Each attribute row therefore moves through HBM once (read fp32, written
// as int32 coefficients) plus once more per extra phase it is pending in.  The schedule (phase lists,
// per-tile merge records sorted by level, a/b factors) is built once from the Morton codes by a keys-only
// cooperative kernel -- the paper's "prelude" -- and is shared by the forward and the inverse transform.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace gsnfs {

constexpr int T = kRahtTile;

struct QStepParams {
  float step[GSNFS_MAX_CHANNELS];
};

__device__ __forceinline__ uint32_t lower_bound_u64(const uint64_t* a, uint32_t lo, uint32_t hi, uint64_t x) {
  while (lo < hi) {                      // first index in [lo, hi) with a[idx] >= x, else hi
    const uint32_t mid = (lo + hi) >> 1;
    if (a[mid] < x) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// ------------------------------------------------------------------------------------------------
// Schedule ("prelude"): all phases in one cooperative launch.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) raht_schedule_kernel(
    const uint64_t* __restrict__ keys, const uint32_t* __restrict__ P, uint32_t n_host,
    const uint32_t* __restrict__ n_dev, uint32_t* __restrict__ idx_pool, uint4* __restrict__ rec,
    RahtTileHdr* __restrict__ hdr, uint32_t* __restrict__ tile_pend, RahtPlan* __restrict__ plan,
    uint32_t pool_rows, uint32_t hdr_cap) {
  cg::grid_group grid = cg::this_grid();
  __shared__ uint64_t s_key[T];
  __shared__ uint32_t s_vidx[T + 1];
  __shared__ uint16_t s_wl[8][64];
  __shared__ uint32_t s_tot[64];
  __shared__ uint32_t s_lstart[64];
  __shared__ uint32_t s_pmask[8];
  __shared__ uint64_t s_edge[2];
  __shared__ uint32_t s_red[9];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t Nv = n_dev ? min(*n_dev, n_host) : n_host;
  uint32_t M = Nv, poff = 0, toff = 0;
  int p = 1;
  if (blockIdx.x == 0 && tid == 0) {
    plan->M[1] = Nv; plan->poff[1] = 0; plan->toff[1] = 0; plan->overflow = 0; plan->nphases = 1;
  }
  while (true) {
    const uint32_t ntiles = (M + T - 1) / T;
    const uint32_t poff_next = (p == 1) ? 0u : poff + M;
    const uint32_t* idx_p = (p == 1) ? nullptr : idx_pool + poff;
    if (toff + ntiles > hdr_cap) {               // uniform over the grid
      if (blockIdx.x == 0 && tid == 0) plan->overflow = 1;
      break;
    }
    if (blockIdx.x == 0 && tid == 0) { plan->M[p + 1] = 0; plan->poff[p + 1] = poff_next; plan->toff[p + 1] = toff + ntiles; }

    // ---- step A: per tile, find the butterflies local to the tile and sort them by level
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const uint32_t ks = tile * T;
      const uint32_t cnt = min((uint32_t)T, M - ks);
      const bool valid = (uint32_t)tid < cnt;
      const uint32_t vidx = valid ? (idx_p ? idx_p[ks + tid] : ks + tid) : 0xffffffffu;
      const uint64_t mk = valid ? keys[vidx] : ~0ull;
      s_key[tid] = mk;
      if (valid) s_vidx[tid] = vidx;                 // slot cnt is written by thread 0 below
      for (int i = tid; i < 8 * 64; i += 256) (&s_wl[0][0])[i] = 0;
      if (tid == 0) {
        const bool has_next = ks + cnt < M;
        const uint32_t vend = has_next ? (idx_p ? idx_p[ks + cnt] : ks + cnt) : Nv;
        s_vidx[cnt] = vend;                                        // cnt <= T: slot T exists
        s_edge[0] = ks > 0 ? keys[idx_p ? idx_p[ks - 1] : ks - 1] : 0ull;
        s_edge[1] = has_next ? keys[vend] : 0ull;
      }
      __syncthreads();
      const bool has_prev = ks > 0, has_next = ks + cnt < M;
      const uint64_t x_first = s_edge[0] ^ s_key[0];
      const uint64_t x_end = s_edge[1] ^ s_key[cnt - 1];
      const int hfirst = has_prev ? (x_first ? msb64(x_first) : 0) : 64;
      const int hend = has_next ? (x_end ? msb64(x_end) : 0) : 64;
      bool local = false;
      int level = 0;
      uint32_t l = 0;
      float fa = 0.f, fb = 0.f;
      if (valid && tid > 0) {
        const uint64_t x = s_key[tid - 1] ^ mk;
        const int h = x ? msb64(x) : 0;                            // x == 0 only for invalid (non-unique) input
        const uint64_t lowp = (mk >> (h + 1)) << (h + 1);
        const uint64_t hip = ((mk >> h) + 1ull) << h;
        l = lower_bound_u64(s_key, 0, tid, lowp);
        const uint32_t r = lower_bound_u64(s_key, tid + 1, cnt, hip);
        local = (l > 0 || hfirst > h) && (r < cnt || hend > h);
        if (local) {
          level = h + 1;
          const uint32_t vk = s_vidx[tid], vl = s_vidx[l], vr = s_vidx[r];
          const double w0 = P ? (double)(P[vk] - P[vl]) : (double)(vk - vl);
          const double w1 = P ? (double)(P[vr] - P[vk]) : (double)(vr - vk);
          fa = (float)sqrt(w0 / (w0 + w1));
          fb = (float)sqrt(w1 / (w0 + w1));
        }
      }
      // rank among the tile's butterflies of the same level (warp match, then prefix over warps)
      const unsigned peers = __match_any_sync(0xffffffffu, level);
      const unsigned lt = peers & lanemask_lt();
      if (local && lt == 0) s_wl[warp][level - 1] = (uint16_t)__popc(peers);
      const unsigned pend_b = __ballot_sync(0xffffffffu, valid && !local);
      if (lane == 0) s_pmask[warp] = pend_b;
      __syncthreads();
      if (tid < 64) {
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) { const uint32_t c = s_wl[w][tid]; s_wl[w][tid] = (uint16_t)run; run += c; }
        s_tot[tid] = run;
      }
      __syncthreads();
      if (warp == 0) {                                             // exclusive scan of 64 level totals
        const uint32_t t0 = s_tot[2 * lane], t1 = s_tot[2 * lane + 1];
        uint32_t inc = t0 + t1;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
        const uint32_t ex = inc - (t0 + t1);
        s_lstart[2 * lane] = ex;
        s_lstart[2 * lane + 1] = ex + t0;
      }
      __syncthreads();
      RahtTileHdr* h_out = hdr + toff + tile;
      if (local) {
        const uint32_t j = s_lstart[level - 1] + s_wl[warp][level - 1] + __popc(lt);
        uint4 rr;
        rr.x = (uint32_t)tid | (l << 8) | ((uint32_t)level << 16);
        rr.y = __float_as_uint(fa);
        rr.z = __float_as_uint(fb);
        rr.w = vidx;
        rec[(size_t)(toff + tile) * T + j] = rr;
      }
      if (tid < 64) h_out->lev_end[tid] = (uint16_t)(s_lstart[tid] + s_tot[tid]);
      if (tid < 8) h_out->pendmask[tid] = s_pmask[tid];
      if (tid == 0) {
        uint32_t np = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) np += __popc(s_pmask[w]);
        h_out->npend = np;
        h_out->nent = cnt;
        h_out->nmerge = cnt - np;
        h_out->pend_off = 0;
        tile_pend[tile] = np;
      }
      __syncthreads();
    }
    grid.sync();

    // ---- step B: offsets of the pending entries, next phase's index list
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      uint32_t part = 0;
      for (uint32_t t = tid; t < tile; t += 256) part += tile_pend[t];
      part = __reduce_add_sync(0xffffffffu, part);
      if (lane == 0) s_red[warp] = part;
      if (tid < 8) s_pmask[tid] = hdr[toff + tile].pendmask[tid];
      __syncthreads();
      uint32_t pend_off = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) pend_off += s_red[w];
      uint32_t before = 0, np = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) { const uint32_t c = __popc(s_pmask[w]); if (w < warp) before += c; np += c; }
      const uint32_t ks = tile * T;
      const bool pend = (s_pmask[warp] >> lane) & 1u;
      const bool fits = (uint64_t)poff_next + pend_off + np <= pool_rows;
      if (pend && fits) {
        const uint32_t rank = before + __popc(s_pmask[warp] & lanemask_lt());
        idx_pool[poff_next + pend_off + rank] = idx_p ? idx_p[ks + tid] : ks + tid;
      }
      if (tid == 0) {
        hdr[toff + tile].pend_off = pend_off;
        if (!fits) plan->overflow = 1;
        if (tile == ntiles - 1) plan->M[p + 1] = pend_off + np;
      }
      __syncthreads();
    }
    grid.sync();
    const uint32_t M_next = *((volatile uint32_t*)&plan->M[p + 1]);
    const uint32_t ovf = *((volatile uint32_t*)&plan->overflow);
    if (M_next <= 1 || ovf || p + 1 > kRahtMaxPhases) break;
    poff = poff_next;
    toff += ntiles;
    M = M_next;
    ++p;
  }
  if (blockIdx.x == 0 && tid == 0) plan->nphases = (uint32_t)p;
}

// ------------------------------------------------------------------------------------------------
// Transform kernels.  VEC = 4: channels % 4 == 0 (float4 rows);  VEC = 1: any channel count.
// A butterfly is handled by a half-warp (16 lanes x VEC channels per step).
// ------------------------------------------------------------------------------------------------
template <int VEC> struct RowVec;
template <> struct RowVec<4> { using type = float4; };
template <> struct RowVec<1> { using type = float; };

__device__ __forceinline__ float4 bf_lo(float a, float b, float4 y0, float4 y1) {
  return make_float4(fmaf(a, y0.x, b * y1.x), fmaf(a, y0.y, b * y1.y), fmaf(a, y0.z, b * y1.z), fmaf(a, y0.w, b * y1.w));
}
__device__ __forceinline__ float4 bf_hi(float a, float b, float4 y0, float4 y1) {
  return make_float4(fmaf(a, y1.x, -b * y0.x), fmaf(a, y1.y, -b * y0.y), fmaf(a, y1.z, -b * y0.z), fmaf(a, y1.w, -b * y0.w));
}
__device__ __forceinline__ float bf_lo(float a, float b, float y0, float y1) { return fmaf(a, y0, b * y1); }
__device__ __forceinline__ float bf_hi(float a, float b, float y0, float y1) { return fmaf(a, y1, -b * y0); }
__device__ __forceinline__ float4 vscale(float4 v, double s) {
  return make_float4((float)((double)v.x * s), (float)((double)v.y * s), (float)((double)v.z * s), (float)((double)v.w * s));
}
__device__ __forceinline__ float vscale(float v, double s) { return (float)((double)v * s); }

__device__ __forceinline__ int quant1(float y, double inv, double f) {
  double m = floor(fma(fabs((double)y), inv, f));
  m = fmin(m, 2147483647.0);
  const int q = (int)m;
  return y < 0.f ? -q : q;
}
__device__ __forceinline__ float dequant1(int q, double step, double bias) {
  if (q == 0) return 0.f;
  const double m = fabs((double)q) + bias;
  return (float)(q < 0 ? -m * step : m * step);
}

template <int VEC>
__device__ __forceinline__ void store_coeff(const float* row_s, int c, int C, size_t orow, const double* s_qinv,
                                            double dz, int32_t* out_q, float* out_f) {
  if constexpr (VEC == 4) {
    const float4 y = reinterpret_cast<const float4*>(row_s)[c];
    if (out_f) reinterpret_cast<float4*>(out_f + orow * C)[c] = y;
    if (out_q) {
      int4 q;
      q.x = quant1(y.x, s_qinv[4 * c + 0], dz); q.y = quant1(y.y, s_qinv[4 * c + 1], dz);
      q.z = quant1(y.z, s_qinv[4 * c + 2], dz); q.w = quant1(y.w, s_qinv[4 * c + 3], dz);
      reinterpret_cast<int4*>(out_q + orow * C)[c] = q;
    }
  } else {
    const float y = row_s[c];
    if (out_f) out_f[orow * C + c] = y;
    if (out_q) out_q[orow * C + c] = quant1(y, s_qinv[c], dz);
  }
}

template <int VEC>
__global__ void __launch_bounds__(256) raht_forward_kernel(
    const float* __restrict__ attr_in, const uint32_t* __restrict__ weights, float* __restrict__ pool,
    const uint4* __restrict__ rec, const RahtTileHdr* __restrict__ hdr, const RahtPlan* __restrict__ plan, int C,
    int levels, QStepParams qs, int has_q, double dz, int32_t* __restrict__ out_q, float* __restrict__ out_f) {
  using V = typename RowVec<VEC>::type;
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) unsigned char s_dyn[];
  float* s_rows = reinterpret_cast<float*>(s_dyn);                      // T x C
  double* s_qinv = reinterpret_cast<double*>(s_dyn + sizeof(float) * T * C);   // C
  __shared__ uint4 s_rec[T];
  __shared__ RahtTileHdr s_hdr;
  __shared__ uint16_t s_plist[T];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int hw = tid >> 4, l16 = tid & 15;
  const int cv = C / VEC;
  for (int c = tid; c < C; c += 256) s_qinv[c] = has_q ? 1.0 / (double)qs.step[c] : 0.0;
  if (!has_q) out_q = nullptr;
  const uint32_t nph = plan->nphases;
  if (plan->overflow) return;                                           // uniform: no grid.sync mismatch
  for (uint32_t p = 1; p <= nph; ++p) {
    const uint32_t M = plan->M[p], Mnext = plan->M[p + 1];
    const uint32_t ntiles = (M + T - 1) / T, toff = plan->toff[p];
    const float* src = (p == 1) ? attr_in : pool + (size_t)plan->poff[p] * C;
    float* dstp = pool + (size_t)plan->poff[p + 1] * C;
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const uint32_t ks = tile * T;
      if (tid < (int)(sizeof(RahtTileHdr) / 4))
        reinterpret_cast<uint32_t*>(&s_hdr)[tid] = reinterpret_cast<const uint32_t*>(hdr + toff + tile)[tid];
      __syncthreads();
      const uint32_t nent = s_hdr.nent, nmerge = s_hdr.nmerge, npend = s_hdr.npend;
      if ((uint32_t)tid < nmerge) s_rec[tid] = rec[(size_t)(toff + tile) * T + tid];
      {
        const V* g = reinterpret_cast<const V*>(src + (size_t)ks * C);
        V* s = reinterpret_cast<V*>(s_rows);
        const uint32_t tot = nent * cv;
        for (uint32_t i = tid; i < tot; i += 256) s[i] = g[i];
      }
      {   // list of pending entries in order
        const uint32_t pm = s_hdr.pendmask[warp];
        uint32_t before = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) if (w < warp) before += __popc(s_hdr.pendmask[w]);
        if ((pm >> lane) & 1u) s_plist[before + __popc(pm & lanemask_lt())] = (uint16_t)tid;
      }
      __syncthreads();
      if (p == 1 && weights) {                                          // [R2] x_i = sqrt(w_i) a_i
        for (uint32_t k = hw; k < nent; k += 16) {
          const uint32_t w = weights[ks + k];
          if (w != 1u) {
            const double sw = sqrt((double)w);
            V* r = reinterpret_cast<V*>(s_rows + (size_t)k * C);
            for (int c = l16; c < cv; c += 16) r[c] = vscale(r[c], sw);
          }
        }
        __syncthreads();
      }
      uint32_t sj = 0;
      for (int l = 1; l <= levels; ++l) {
        const uint32_t ej = s_hdr.lev_end[l - 1];
        if (ej > sj) {
          for (uint32_t j = sj + hw; j < ej; j += 16) {
            const uint4 rr = s_rec[j];
            const uint32_t k = rr.x & 0xffu, li = (rr.x >> 8) & 0xffu;
            const float a = __uint_as_float(rr.y), b = __uint_as_float(rr.z);
            V* r0 = reinterpret_cast<V*>(s_rows + (size_t)li * C);
            V* r1 = reinterpret_cast<V*>(s_rows + (size_t)k * C);
            for (int c = l16; c < cv; c += 16) {
              const V y0 = r0[c], y1 = r1[c];
              r0[c] = bf_lo(a, b, y0, y1);                               // low-pass stays at the left index
              r1[c] = bf_hi(a, b, y0, y1);                               // high-pass at the right index
            }
          }
          __syncthreads();
        }
        sj = ej;
      }
      // finished high-pass coefficients -> canonical rows of the output
      for (uint32_t j = hw; j < nmerge; j += 16) {
        const uint4 rr = s_rec[j];
        const uint32_t k = rr.x & 0xffu;
        for (int c = l16; c < cv; c += 16)
          store_coeff<VEC>(s_rows + (size_t)k * C, c, C, (size_t)rr.w, s_qinv, dz, out_q, out_f);
      }
      // pending low-pass nodes -> next phase's row pool (or, when one node is left, the DC at row 0)
      const uint32_t pend_off = s_hdr.pend_off;
      for (uint32_t j = hw; j < npend; j += 16) {
        const uint32_t k = s_plist[j];
        if (Mnext == 1u) {
          for (int c = l16; c < cv; c += 16)
            store_coeff<VEC>(s_rows + (size_t)k * C, c, C, (size_t)0, s_qinv, dz, out_q, out_f);
        } else {
          const V* r = reinterpret_cast<const V*>(s_rows + (size_t)k * C);
          V* d = reinterpret_cast<V*>(dstp + (size_t)(pend_off + j) * C);
          for (int c = l16; c < cv; c += 16) d[c] = r[c];
        }
      }
      __syncthreads();
    }
    if (p < nph) grid.sync();
  }
}

template <int VEC>
__device__ __forceinline__ void load_coeff(float* row_s, int c, int C, size_t irow, const double* s_step, double bias,
                                           const int32_t* in_q, const float* in_f) {
  if constexpr (VEC == 4) {
    float4 y;
    if (in_q) {
      const int4 q = reinterpret_cast<const int4*>(in_q + irow * C)[c];
      y = make_float4(dequant1(q.x, s_step[4 * c + 0], bias), dequant1(q.y, s_step[4 * c + 1], bias),
                      dequant1(q.z, s_step[4 * c + 2], bias), dequant1(q.w, s_step[4 * c + 3], bias));
    } else {
      y = reinterpret_cast<const float4*>(in_f + irow * C)[c];
    }
    reinterpret_cast<float4*>(row_s)[c] = y;
  } else {
    row_s[c] = in_q ? dequant1(in_q[irow * C + c], s_step[c], bias) : in_f[irow * C + c];
  }
}

template <int VEC>
__global__ void __launch_bounds__(256) raht_inverse_kernel(
    const int32_t* __restrict__ in_q, const float* __restrict__ in_f, const uint32_t* __restrict__ weights,
    float* __restrict__ pool, const uint4* __restrict__ rec, const RahtTileHdr* __restrict__ hdr,
    const RahtPlan* __restrict__ plan, int C, int levels, QStepParams qs, double bias, float* __restrict__ attr_out) {
  using V = typename RowVec<VEC>::type;
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) unsigned char s_dyn[];
  float* s_rows = reinterpret_cast<float*>(s_dyn);
  double* s_step = reinterpret_cast<double*>(s_dyn + sizeof(float) * T * C);
  __shared__ uint4 s_rec[T];
  __shared__ RahtTileHdr s_hdr;
  __shared__ uint16_t s_plist[T];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int hw = tid >> 4, l16 = tid & 15;
  const int cv = C / VEC;
  for (int c = tid; c < C; c += 256) s_step[c] = in_q ? (double)qs.step[c] : 0.0;
  const uint32_t nph = plan->nphases;
  if (plan->overflow) return;
  for (uint32_t p = nph; p >= 1; --p) {
    const uint32_t M = plan->M[p], Mnext = plan->M[p + 1];
    const uint32_t ntiles = (M + T - 1) / T, toff = plan->toff[p];
    const float* srcp = pool + (size_t)plan->poff[p + 1] * C;            // low-pass values from phase p+1
    float* dst = (p == 1) ? attr_out : pool + (size_t)plan->poff[p] * C;
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const uint32_t ks = tile * T;
      if (tid < (int)(sizeof(RahtTileHdr) / 4))
        reinterpret_cast<uint32_t*>(&s_hdr)[tid] = reinterpret_cast<const uint32_t*>(hdr + toff + tile)[tid];
      __syncthreads();
      const uint32_t nent = s_hdr.nent, nmerge = s_hdr.nmerge, npend = s_hdr.npend;
      if ((uint32_t)tid < nmerge) s_rec[tid] = rec[(size_t)(toff + tile) * T + tid];
      {
        const uint32_t pm = s_hdr.pendmask[warp];
        uint32_t before = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) if (w < warp) before += __popc(s_hdr.pendmask[w]);
        if ((pm >> lane) & 1u) s_plist[before + __popc(pm & lanemask_lt())] = (uint16_t)tid;
      }
      __syncthreads();
      for (uint32_t j = hw; j < nmerge; j += 16) {                       // high-pass coefficients of this phase
        const uint4 rr = s_rec[j];
        const uint32_t k = rr.x & 0xffu;
        for (int c = l16; c < cv; c += 16)
          load_coeff<VEC>(s_rows + (size_t)k * C, c, C, (size_t)rr.w, s_step, bias, in_q, in_f);
      }
      const uint32_t pend_off = s_hdr.pend_off;
      for (uint32_t j = hw; j < npend; j += 16) {                        // low-pass inputs
        const uint32_t k = s_plist[j];
        if (Mnext == 1u) {
          for (int c = l16; c < cv; c += 16)
            load_coeff<VEC>(s_rows + (size_t)k * C, c, C, (size_t)0, s_step, bias, in_q, in_f);
        } else {
          const V* g = reinterpret_cast<const V*>(srcp + (size_t)(pend_off + j) * C);
          V* r = reinterpret_cast<V*>(s_rows + (size_t)k * C);
          for (int c = l16; c < cv; c += 16) r[c] = g[c];
        }
      }
      __syncthreads();
      for (int l = levels; l >= 1; --l) {
        const uint32_t ej = s_hdr.lev_end[l - 1];
        const uint32_t sj = l >= 2 ? s_hdr.lev_end[l - 2] : 0u;
        if (ej > sj) {
          for (uint32_t j = sj + hw; j < ej; j += 16) {
            const uint4 rr = s_rec[j];
            const uint32_t k = rr.x & 0xffu, li = (rr.x >> 8) & 0xffu;
            const float a = __uint_as_float(rr.y), b = __uint_as_float(rr.z);
            V* r0 = reinterpret_cast<V*>(s_rows + (size_t)li * C);
            V* r1 = reinterpret_cast<V*>(s_rows + (size_t)k * C);
            for (int c = l16; c < cv; c += 16) {
              const V y0 = r0[c], y1 = r1[c];
              r0[c] = bf_hi(a, b, y1, y0);          // a*y0 - b*y1  (A.6 l.37)
              r1[c] = bf_lo(b, a, y0, y1);          // b*y0 + a*y1  (A.6 l.38)
            }
          }
          __syncthreads();
        }
      }
      if (p == 1 && weights) {                                           // [R2] a_i = x_i / sqrt(w_i)
        for (uint32_t k = hw; k < nent; k += 16) {
          const uint32_t w = weights[ks + k];
          if (w != 1u) {
            const double sw = 1.0 / sqrt((double)w);
            V* r = reinterpret_cast<V*>(s_rows + (size_t)k * C);
            for (int c = l16; c < cv; c += 16) r[c] = vscale(r[c], sw);
          }
        }
        __syncthreads();
      }
      {
        V* g = reinterpret_cast<V*>(dst + (size_t)ks * C);
        const V* s = reinterpret_cast<const V*>(s_rows);
        const uint32_t tot = nent * cv;
        for (uint32_t i = tid; i < tot; i += 256) g[i] = s[i];
      }
      __syncthreads();
    }
    if (p > 1) grid.sync();
  }
}

// ------------------------------------------------------------------------------------------------
static size_t raht_smem_bytes(int C) { return sizeof(float) * (size_t)T * C + sizeof(double) * C; }

int raht_setup(gsnfs_ctx* ctx) {
  const size_t smem = raht_smem_bytes(ctx->max_channels);
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_forward_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_forward_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_inverse_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_inverse_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  return GSNFS_OK;
}

template <typename K>
static int coop_grid(gsnfs_ctx* ctx, K kernel, size_t smem, uint32_t want, int* out) {
  int per_sm = 0;
  GSNFS_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, 256, smem));
  if (per_sm < 1) { snprintf(ctx->err, sizeof(ctx->err), "raht kernel does not fit on an SM"); return GSNFS_E_CUDA; }
  const uint32_t cap = (uint32_t)per_sm * (uint32_t)ctx->num_sms;
  *out = (int)max(1u, min(cap, want));
  return GSNFS_OK;
}

int run_raht(gsnfs_ctx* ctx, cudaStream_t st, bool inverse, const uint64_t* d_keys, const uint32_t* d_weights,
             uint32_t n_voxels, const gsnfs_counts* d_counts, int depth, const float* d_in_f, const int32_t* d_in_q,
             int channels, const float* qstep, const gsnfs_quant* quant, int32_t* d_out_q, float* d_out_f) {
  if (n_voxels == 0) return GSNFS_OK;
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const uint32_t* P = nullptr;
  if (d_weights) {
    int rc = run_scan_u32(ctx, st, d_weights, ctx->wprefix, n_voxels, n_dev);
    if (rc != GSNFS_OK) return rc;
    P = ctx->wprefix;
  }
  const uint32_t want = (n_voxels + T - 1) / T;
  uint32_t pool_rows = (uint32_t)ctx->raht_pool_rows, hdr_cap = (uint32_t)ctx->raht_hdr_cap;
  {
    int grid = 0;
    int rc = coop_grid(ctx, raht_schedule_kernel, 0, want, &grid);
    if (rc != GSNFS_OK) return rc;
    void* args[] = {(void*)&d_keys, (void*)&P, (void*)&n_voxels, (void*)&n_dev, (void*)&ctx->raht_idx,
                    (void*)&ctx->raht_rec, (void*)&ctx->raht_hdr, (void*)&ctx->raht_tile_pend, (void*)&ctx->raht_plan,
                    (void*)&pool_rows, (void*)&hdr_cap};
    GSNFS_KERNEL(ctx, st, "raht_schedule");
    GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel((void*)raht_schedule_kernel, dim3(grid), dim3(256), args, 0, st));
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  QStepParams qs;
  for (int c = 0; c < GSNFS_MAX_CHANNELS; ++c) qs.step[c] = (qstep && c < channels) ? qstep[c] : 1.0f;
  const double dz = quant ? (double)quant->dz_round : (double)(1.0f / 3.0f);
  const double bias = quant ? (double)quant->recon_bias : 0.0;
  const size_t smem = raht_smem_bytes(channels);
  const int levels = 3 * depth;
  const bool vec4 = (channels % 4) == 0;
  int grid = 0;
  if (!inverse) {
    int has_q = (qstep != nullptr && d_out_q != nullptr) ? 1 : 0;
    void* args[] = {(void*)&d_in_f, (void*)&d_weights, (void*)&ctx->raht_rows, (void*)&ctx->raht_rec, (void*)&ctx->raht_hdr,
                    (void*)&ctx->raht_plan, (void*)&channels, (void*)&levels, (void*)&qs, (void*)&has_q, (void*)&dz,
                    (void*)&d_out_q, (void*)&d_out_f};
    void* fn = vec4 ? (void*)raht_forward_kernel<4> : (void*)raht_forward_kernel<1>;
    int rc = vec4 ? coop_grid(ctx, raht_forward_kernel<4>, smem, want, &grid) : coop_grid(ctx, raht_forward_kernel<1>, smem, want, &grid);
    if (rc != GSNFS_OK) return rc;
    GSNFS_KERNEL(ctx, st, "raht_forward");
    GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(256), args, smem, st));
    GSNFS_LAUNCH_CHECK(ctx, st);
  } else {
    void* args[] = {(void*)&d_in_q, (void*)&d_in_f, (void*)&d_weights, (void*)&ctx->raht_rows, (void*)&ctx->raht_rec,
                    (void*)&ctx->raht_hdr, (void*)&ctx->raht_plan, (void*)&channels, (void*)&levels, (void*)&qs, (void*)&bias,
                    (void*)&d_out_f};
    void* fn = vec4 ? (void*)raht_inverse_kernel<4> : (void*)raht_inverse_kernel<1>;
    int rc = vec4 ? coop_grid(ctx, raht_inverse_kernel<4>, smem, want, &grid) : coop_grid(ctx, raht_inverse_kernel<1>, smem, want, &grid);
    if (rc != GSNFS_OK) return rc;
    GSNFS_KERNEL(ctx, st, "raht_inverse");
    GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(256), args, smem, st));
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  return GSNFS_OK;
}

}  // namespace gsnfs
