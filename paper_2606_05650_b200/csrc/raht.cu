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

#include "merge_long.cuh"
#include "raht_math.cuh"

namespace cg = cooperative_groups;

namespace gsnfs {

constexpr int T = kRahtTile;
#ifndef RAHT_XT
#define RAHT_XT 256
#endif
constexpr int kXT = RAHT_XT;        // threads per CTA of the transform kernels

// ------------------------------------------------------------------------------------------------
// Transform kernels.  VEC = 4: channels % 4 == 0 (float4 rows);  VEC = 1: any channel count.
// A butterfly is handled by a half-warp (16 lanes x VEC channels per step).
// ------------------------------------------------------------------------------------------------
// Per-tile metadata staged in shared memory (double buffered: the next tile's is prefetched).
struct __align__(16) TileMeta {
  uint4 rec[T];
  RahtTileHdr hdr;
  uint32_t w[T];          // leaf weights of the tile's rows (phase 1 with weights only)
  uint32_t g[T];          // fused merge: first Gaussian of each voxel (phase 1 only)
};

__device__ __forceinline__ void prefetch_meta(TileMeta* m, const uint4* rec, const RahtTileHdr* hdr,
                                              const uint32_t* weights, const uint32_t* gsrc, size_t tglob, uint32_t ks,
                                              uint32_t cnt) {
  const int tid = threadIdx.x;
  if (tid < T) cp_async16(&m->rec[tid], rec + tglob * T + tid);
  if (tid < (int)(sizeof(RahtTileHdr) / 16))
    cp_async16(reinterpret_cast<uint4*>(&m->hdr) + tid, reinterpret_cast<const uint4*>(hdr + tglob) + tid);
  if (weights && (uint32_t)tid < cnt) cp_async4(&m->w[tid], weights + ks + tid);
  if (gsrc && (uint32_t)tid < cnt) cp_async4(&m->g[tid], gsrc + ks + tid);
}

template <int VEC>
__device__ __forceinline__ void stage_rows_contig(float* s_rows, const float* src, uint32_t nrows, int C) {
  if constexpr (VEC == 4) {
    const uint32_t tot = nrows * (uint32_t)(C / 4);
    const float4* g = reinterpret_cast<const float4*>(src);
    float4* s = reinterpret_cast<float4*>(s_rows);
    for (uint32_t i = threadIdx.x; i < tot; i += kXT) cp_async16(s + i, g + i);
  } else {
    const uint32_t tot = nrows * (uint32_t)C;
    for (uint32_t i = threadIdx.x; i < tot; i += kXT) cp_async4(s_rows + i, src + i);
  }
}

struct GatherArgs {          // fused merge: rows of phase 1 are gathered through the sorted permutation
  const uint32_t* gsrc;      // NULL => rows are contiguous
  const uint32_t* perm;
  const uint32_t* vstart;
  double* partial;           // chunk partial sums of the long runs (merge_long.cuh)
};

template <int VEC>
__global__ void __launch_bounds__(kXT, 3) raht_forward_kernel(
    const float* __restrict__ attr_in, const uint32_t* __restrict__ weights, GatherArgs ga, float* __restrict__ pool,
    const uint4* __restrict__ rec, const RahtTileHdr* __restrict__ hdr, RahtPlan* __restrict__ plan, int C,
    QStepParams qs, int has_q, double dz, int32_t* __restrict__ out_q, float* __restrict__ out_f) {
  using V = typename RowVec<VEC>::type;
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) unsigned char s_dyn[];
  float* s_rows = reinterpret_cast<float*>(s_dyn);                                // T x C
  TileMeta* s_meta = reinterpret_cast<TileMeta*>(s_dyn + sizeof(float) * T * C);  // x 2
  QuantTab qt;
  qt.inv64 = reinterpret_cast<double*>(s_dyn + sizeof(float) * T * C + 2 * sizeof(TileMeta));
  qt.inv32 = reinterpret_cast<float*>(qt.inv64 + ((C + 3) & ~3));
  __shared__ uint32_t s_dst[T];     // destination row: out row (finished) or pool row | 0x80000000 (pending)

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cv = C / VEC;
  // lanes per row: the smallest power of two >= cv, at most 16 (C = 56: a half-warp per row; C = 3: four lanes per row,
  // eight butterflies per warp step)
  int lsh = 4;
  while (lsh > 0 && (1 << (lsh - 1)) >= cv) --lsh;
  const int lpr = 1 << lsh, nhw = kXT >> lsh;
  const int hw = tid >> lsh, l16 = tid & (lpr - 1);
  for (int c = tid; c < C; c += kXT) {
    const double iv = has_q ? 1.0 / (double)qs.step[c] : 0.0;
    qt.inv64[c] = iv;
    qt.inv32[c] = (float)iv;
  }
  const float dz32 = (float)(dz - 0.5);                                  // the quantiser's half-shifted rounding offset
  const uint32_t cv_magic = make_div_magic((uint32_t)(C / VEC));
  if (!has_q) out_q = nullptr;
  const uint32_t nph = plan->nphases;
  if (plan->overflow) return;                                           // uniform: no grid.sync mismatch
  if (ga.gsrc && plan->has_long) {       // fused merge with long duplicate runs: chunk partial sums by the whole grid first
    const uint32_t nv = plan->M[1];
    const uint32_t nchunks = (ga.vstart[nv] + kLongChunk - 1) / kLongChunk;
    for (uint32_t chunk = blockIdx.x * nhw + hw; chunk < nchunks; chunk += gridDim.x * nhw)
      long_chunk_partials<VEC>(attr_in, C, ga.perm, ga.vstart, nv, chunk, ga.partial, l16, lpr);
    __threadfence();
    grid.sync();
  }
  for (uint32_t p = 1; p <= nph; ++p) {
    const uint32_t M = plan->M[p], Mnext = plan->M[p + 1];
    const uint32_t ntiles = (M + T - 1) / T, toff = plan->toff[p];
    const float* src = (p == 1) ? attr_in : pool + (size_t)plan->poff[p] * C;
    float* dstp = pool + (size_t)plan->poff[p + 1] * C;
    const uint32_t* wts = (p == 1) ? weights : nullptr;
    const uint32_t* gsrc = (p == 1) ? ga.gsrc : nullptr;
    int cur = 0;
    if (blockIdx.x < ntiles) {
      const uint32_t ks = blockIdx.x * T;
      prefetch_meta(&s_meta[0], rec, hdr, wts, gsrc, (size_t)toff + blockIdx.x, ks, min((uint32_t)T, M - ks));
    }
    cp_async_commit();
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const uint32_t ks = tile * T;
      const uint32_t nent = min((uint32_t)T, M - ks);
      TileMeta* mt = &s_meta[cur];
      if (gsrc) {
        cp_async_wait_all();                       // meta(cur) was prefetched one tile ago
        __syncthreads();
        const uint32_t tot = nent * (uint32_t)cv;
        for (uint32_t i = tid; i < tot; i += kXT) {
          const uint32_t k = div_cv(i, cv_magic, (uint32_t)cv);
          const uint32_t c = i - k * (uint32_t)cv;
          const float* g = src + (size_t)mt->g[k] * C;
          if constexpr (VEC == 4) cp_async16(s_rows + (size_t)k * C + 4 * c, g + 4 * c);
          else cp_async4(s_rows + (size_t)k * C + c, g + c);
        }
      } else {
        stage_rows_contig<VEC>(s_rows, src + (size_t)ks * C, nent, C);
      }
      cp_async_commit();
      const uint32_t tnext = tile + gridDim.x;
      if (tnext < ntiles) {
        const uint32_t ksn = tnext * T;
        prefetch_meta(&s_meta[cur ^ 1], rec, hdr, wts, gsrc, (size_t)toff + tnext, ksn, min((uint32_t)T, M - ksn));
      }
      cp_async_commit();
      asm volatile("cp.async.wait_group 1;" ::: "memory");      // meta(cur) + rows(cur) landed; meta(next) may be in flight
      __syncthreads();
      const uint32_t nmerge = mt->hdr.nmerge, nseg = (mt->hdr.nent >> 16) & 0x7fu;
      {   // destination of every entry, in natural order
        const uint32_t pm = warp < 8 ? mt->hdr.pendmask[warp] : 0u;
        uint32_t before = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) if (w < warp) before += __popc(mt->hdr.pendmask[w]);
        if ((pm >> lane) & 1u) s_dst[tid] = 0x80000000u | (mt->hdr.pend_off + before + __popc(pm & lanemask_lt()));
        if ((uint32_t)tid < nmerge) { const uint4 rr = mt->rec[tid]; s_dst[rr.x & 0xffu] = rr.w; }
      }
      // [R2] x_i = sqrt(w_i) a_i: only rows with w != 1 need work (block-uniform test first)
      const bool nonunit = (mt->hdr.nent >> 31) != 0u;      // the schedule saw a leaf weight != 1 in this tile
      bool staged = false;             // a barrier has passed since the rows and s_dst were written
      if (wts && nonunit) {
        __syncthreads();
        for (uint32_t k = hw; k < nent; k += nhw) {
          const uint32_t w = mt->w[k];
          if (w != 1u) {
            V* r = reinterpret_cast<V*>(s_rows + (size_t)k * C);
            if (gsrc) {      // duplicate voxel: mean of its Gaussians, fp64 accumulation in sorted order [O9]
              const uint32_t s0 = ga.vstart[ks + k];
              for (int c = l16; c < cv; c += lpr) {
                if (w >= kLongRun) {
                  double a[VEC];
                  long_run_sum<VEC>(ga.partial, C, s0, s0 + w, c, a);
                  const double dw = (double)w;
                  if constexpr (VEC == 4) r[c] = make_float4((float)(a[0] / dw), (float)(a[1] / dw), (float)(a[2] / dw), (float)(a[3] / dw));
                  else r[c] = (float)(a[0] / dw);
                } else if constexpr (VEC == 4) {
                  const float4 x = r[c];
                  double a0 = x.x, a1 = x.y, a2 = x.z, a3 = x.w;
                  uint32_t q = 1;
                  for (; q + 4 <= w; q += 4) {       // four rows in flight; the sums stay in sorted order
                    uint32_t g4[4];
                    float4 y4[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) g4[u] = ga.perm[s0 + q + u];
#pragma unroll
                    for (int u = 0; u < 4; ++u) y4[u] = reinterpret_cast<const float4*>(src + (size_t)g4[u] * C)[c];
#pragma unroll
                    for (int u = 0; u < 4; ++u) { a0 += y4[u].x; a1 += y4[u].y; a2 += y4[u].z; a3 += y4[u].w; }
                  }
                  for (; q < w; ++q) {
                    const float4 y = reinterpret_cast<const float4*>(src + (size_t)ga.perm[s0 + q] * C)[c];
                    a0 += y.x; a1 += y.y; a2 += y.z; a3 += y.w;
                  }
                  const double dw = (double)w;
                  r[c] = make_float4((float)(a0 / dw), (float)(a1 / dw), (float)(a2 / dw), (float)(a3 / dw));
                } else {
                  double a0 = r[c];
                  for (uint32_t q = 1; q < w; ++q) a0 += src[(size_t)ga.perm[s0 + q] * C + c];
                  r[c] = (float)(a0 / (double)w);
                }
              }
            }
            const double sw = sqrt((double)w);
            for (int c = l16; c < cv; c += lpr) r[c] = vscale(r[c], sw);
          }
        }
      }
      if (!staged) __syncthreads();
      uint32_t sj = 0;
      for (uint32_t s = 0; s < nseg; ++s) {                               // non-empty levels, bottom-up
        const uint32_t ej = mt->hdr.lev_end[s];
        for (uint32_t j = sj + hw; j < ej; j += nhw) {
          const uint4 rr = mt->rec[j];
          const uint32_t k = rr.x & 0xffu, li = (rr.x >> 8) & 0xffu;
          const float a = __uint_as_float(rr.y), b = __uint_as_float(rr.z);
          V* r0 = reinterpret_cast<V*>(s_rows + (size_t)li * C);
          V* r1 = reinterpret_cast<V*>(s_rows + (size_t)k * C);
          for (int c = l16; c < cv; c += lpr) {
            const V y0 = r0[c], y1 = r1[c];
            r0[c] = bf_lo(a, b, y0, y1);                                   // low-pass stays at the left index
            r1[c] = bf_hi(a, b, y0, y1);                                   // high-pass at the right index
          }
        }
        __syncthreads();
        sj = ej;
      }
      if (tnext < ntiles) {          // next tile's input rows -> L2 while this tile is written out
        const uint32_t ksn = tnext * T;
        if ((uint32_t)tid < min((uint32_t)T, M - ksn)) {
          if (gsrc) {
            cp_async_wait_all();       // this thread's own piece of meta(next) (its g entry) has landed
            prefetch_row_l2(src + (size_t)s_meta[cur ^ 1].g[tid] * C, C);
          } else {
            prefetch_row_l2(src + (size_t)(ksn + tid) * C, C);
          }
        }
      }
      // rows out, in natural order: finished high-pass -> canonical output row (quantised); pending
      // low-pass -> next phase's row pool, or -- when a single node is left -- the DC at output row 0
      {
        const uint32_t tot = nent * (uint32_t)cv;
        for (uint32_t i = tid; i < tot; i += kXT) {
          const uint32_t k = div_cv(i, cv_magic, (uint32_t)cv);
          const int c = (int)(i - k * (uint32_t)cv);
          const uint32_t d = s_dst[k];
          const float* rs = s_rows + (size_t)k * C;
          if ((d & 0x80000000u) && Mnext != 1u) {
            reinterpret_cast<V*>(dstp + (size_t)(d & 0x7fffffffu) * C)[c] = reinterpret_cast<const V*>(rs)[c];
          } else {
            const size_t orow = (d & 0x80000000u) ? (size_t)0 : (size_t)d;
            store_coeff<VEC>(rs, c, C, orow, qt, dz, dz32, out_q, out_f);
          }
        }
      }
      __syncthreads();
      cur ^= 1;
    }
    cp_async_wait_all();
    if (p < nph) grid.sync();
  }
}

template <int VEC>
__global__ void __launch_bounds__(kXT, 3) raht_inverse_kernel(
    const int32_t* __restrict__ in_q, const float* __restrict__ in_f, const uint32_t* __restrict__ weights,
    float* __restrict__ pool, const uint4* __restrict__ rec, const RahtTileHdr* __restrict__ hdr,
    RahtPlan* __restrict__ plan, int C, QStepParams qs, double bias, float* __restrict__ attr_out) {
  using V = typename RowVec<VEC>::type;
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) unsigned char s_dyn[];
  float* s_rows = reinterpret_cast<float*>(s_dyn);
  TileMeta* s_meta = reinterpret_cast<TileMeta*>(s_dyn + sizeof(float) * T * C);
  QuantTab qt;
  qt.inv64 = reinterpret_cast<double*>(s_dyn + sizeof(float) * T * C + 2 * sizeof(TileMeta));
  qt.inv32 = reinterpret_cast<float*>(qt.inv64 + ((C + 3) & ~3));
  __shared__ uint32_t s_srcrow[T];  // source row: coefficient row (finished) or pool row | 0x80000000 (pending)

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cv = C / VEC;
  // lanes per row: the smallest power of two >= cv, at most 16 (C = 56: a half-warp per row; C = 3: four lanes per row,
  // eight butterflies per warp step)
  int lsh = 4;
  while (lsh > 0 && (1 << (lsh - 1)) >= cv) --lsh;
  const int lpr = 1 << lsh, nhw = kXT >> lsh;
  const int hw = tid >> lsh, l16 = tid & (lpr - 1);
  for (int c = tid; c < C; c += kXT) { qt.inv64[c] = in_q ? (double)qs.step[c] : 0.0; qt.inv32[c] = in_q ? qs.step[c] : 0.f; }
  const uint32_t cv_magic = make_div_magic((uint32_t)(C / VEC));
  const void* coef = in_q ? (const void*)in_q : (const void*)in_f;       // both are 4-byte rows of C entries
  const uint32_t nph = plan->nphases;
  if (plan->overflow) return;
  for (uint32_t p = nph; p >= 1; --p) {
    const uint32_t M = plan->M[p], Mnext = plan->M[p + 1];
    const uint32_t ntiles = (M + T - 1) / T, toff = plan->toff[p];
    const float* srcp = pool + (size_t)plan->poff[p + 1] * C;            // low-pass values from phase p+1
    float* dst = (p == 1) ? attr_out : pool + (size_t)plan->poff[p] * C;
    const uint32_t* wts = (p == 1) ? weights : nullptr;
    int cur = 0;
    if (blockIdx.x < ntiles) {
      const uint32_t ks = blockIdx.x * T;
      prefetch_meta(&s_meta[0], rec, hdr, wts, nullptr, (size_t)toff + blockIdx.x, ks, min((uint32_t)T, M - ks));
    }
    cp_async_commit();
    cp_async_wait_all();
    __syncthreads();
    for (uint32_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const uint32_t ks = tile * T;
      const uint32_t nent = min((uint32_t)T, M - ks);
      TileMeta* mt = &s_meta[cur];
      const uint32_t nmerge = mt->hdr.nmerge, nseg = (mt->hdr.nent >> 16) & 0x7fu;
      {
        const uint32_t pm = warp < 8 ? mt->hdr.pendmask[warp] : 0u;
        uint32_t before = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) if (w < warp) before += __popc(mt->hdr.pendmask[w]);
        if ((pm >> lane) & 1u) s_srcrow[tid] = 0x80000000u | (mt->hdr.pend_off + before + __popc(pm & lanemask_lt()));
        if ((uint32_t)tid < nmerge) { const uint4 rr = mt->rec[tid]; s_srcrow[rr.x & 0xffu] = rr.w; }
      }
      __syncthreads();
      // stage every row of the tile: high-pass coefficients of this phase from the coefficient array,
      // low-pass inputs from phase p+1's rows (or, when a single node is left, the DC = coefficient row 0)
      {
        const uint32_t tot = nent * (uint32_t)cv;
        for (uint32_t i = tid; i < tot; i += kXT) {
          const uint32_t k = div_cv(i, cv_magic, (uint32_t)cv);
          const uint32_t c = i - k * (uint32_t)cv;
          const uint32_t s = s_srcrow[k];
          const float* g = ((s & 0x80000000u) && Mnext != 1u)
                               ? srcp + (size_t)(s & 0x7fffffffu) * C
                               : (const float*)coef + (size_t)((s & 0x80000000u) ? 0u : s) * C;
          if constexpr (VEC == 4) cp_async16(s_rows + (size_t)k * C + 4 * c, g + 4 * c);
          else cp_async4(s_rows + (size_t)k * C + c, g + c);
        }
      }
      cp_async_commit();
      const uint32_t tnext = tile + gridDim.x;
      if (tnext < ntiles) {
        const uint32_t ksn = tnext * T;
        prefetch_meta(&s_meta[cur ^ 1], rec, hdr, wts, nullptr, (size_t)toff + tnext, ksn, min((uint32_t)T, M - ksn));
      }
      cp_async_commit();
      asm volatile("cp.async.wait_group 1;" ::: "memory");
      __syncthreads();
      if (in_q) {                                                          // de-quantise in place
        const uint32_t tot = nent * (uint32_t)cv;
        for (uint32_t i = tid; i < tot; i += kXT) {
          const uint32_t k = div_cv(i, cv_magic, (uint32_t)cv);
          const uint32_t s = s_srcrow[k];
          if (!((s & 0x80000000u) && Mnext != 1u))
            dequant_row_inplace<VEC>(s_rows + (size_t)k * C, (int)(i - k * (uint32_t)cv), qt, bias);
        }
        __syncthreads();
      }
      for (int s = (int)nseg - 1; s >= 0; --s) {                           // non-empty levels, top-down
        const uint32_t ej = mt->hdr.lev_end[s];
        const uint32_t sj = s > 0 ? mt->hdr.lev_end[s - 1] : 0u;
        for (uint32_t j = sj + hw; j < ej; j += nhw) {
          const uint4 rr = mt->rec[j];
          const uint32_t k = rr.x & 0xffu, li = (rr.x >> 8) & 0xffu;
          const float a = __uint_as_float(rr.y), b = __uint_as_float(rr.z);
          V* r0 = reinterpret_cast<V*>(s_rows + (size_t)li * C);
          V* r1 = reinterpret_cast<V*>(s_rows + (size_t)k * C);
          for (int c = l16; c < cv; c += lpr) {
            const V y0 = r0[c], y1 = r1[c];
            r0[c] = bf_hi(a, b, y1, y0);          // a*y0 - b*y1  (A.6 l.37)
            r1[c] = bf_lo(b, a, y0, y1);          // b*y0 + a*y1  (A.6 l.38)
          }
        }
        __syncthreads();
      }
      if (wts && (mt->hdr.nent >> 31) != 0u) {                                   // [R2] a_i = x_i / sqrt(w_i)
        for (uint32_t k = hw; k < nent; k += nhw) {
          const uint32_t w = mt->w[k];
          if (w != 1u) {
            const double sw = 1.0 / sqrt((double)w);
            V* r = reinterpret_cast<V*>(s_rows + (size_t)k * C);
            for (int c = l16; c < cv; c += lpr) r[c] = vscale(r[c], sw);
          }
        }
        __syncthreads();
      }
      if constexpr (VEC == 4) {        // the tile's rows are contiguous in dst: one TMA bulk store
        fence_proxy_async();           // this thread's writes to the staged rows -> visible to the async proxy
        cp_async_wait_all();           // meta(next) before it is read
        __syncthreads();
        if (tid == 0) {
          bulk_s2g(dst + (size_t)ks * C, smem_u32(s_rows), nent * (uint32_t)C * 4u);
          bulk_commit();
          bulk_wait_read();            // the rows have left shared memory: the next tile may be staged over them
        }
      } else {
        V* g = reinterpret_cast<V*>(dst + (size_t)ks * C);
        const V* s = reinterpret_cast<const V*>(s_rows);
        const uint32_t tot = nent * cv;
        for (uint32_t i = tid; i < tot; i += kXT) g[i] = s[i];
        cp_async_wait_all();                                                // meta(next) before it is read
      }
      __syncthreads();
      cur ^= 1;
    }
    if (p > 1) {
      if constexpr (VEC == 4) {        // pool rows written by the async proxy: complete and ordered before the grid barrier
        if (tid == 0) { bulk_wait_all(); fence_proxy_async_all(); }
      }
      grid.sync();
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Quantise an N_v x C fp32 coefficient tensor with one step per channel (one ladder rung from a shared
// transform, section 3.4 L255 + L47-49 bitrate ladder).  Same quantiser as the fused one [R10].
// ------------------------------------------------------------------------------------------------
template <int VEC>
__global__ void __launch_bounds__(256) quantize_kernel(const float* __restrict__ coeff, uint32_t n_host,
                                                       const uint32_t* __restrict__ n_dev, int C, QStepParams qs, double dz,
                                                       int32_t* __restrict__ out_q) {
  __shared__ double s_inv64[(GSNFS_MAX_CHANNELS + 3) & ~3];
  __shared__ __align__(16) float s_inv32[(GSNFS_MAX_CHANNELS + 3) & ~3];
  for (int c = threadIdx.x; c < ((C + 3) & ~3); c += 256) {
    const double iv = c < C ? 1.0 / (double)qs.step[c] : 0.0;
    s_inv64[c] = iv;
    s_inv32[c] = (float)iv;
  }
  __syncthreads();
  QuantTab qt;
  qt.inv64 = s_inv64;
  qt.inv32 = s_inv32;
  const float dz32 = (float)(dz - 0.5);
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const uint32_t cv = (uint32_t)(C / VEC);
  const uint64_t tot = (uint64_t)n * cv;
  const uint64_t stride = (uint64_t)gridDim.x * 256u;
  for (uint64_t i = (uint64_t)blockIdx.x * 256u + threadIdx.x; i < tot; i += stride) {
    const int c = (int)(i % cv);
    if constexpr (VEC == 4) reinterpret_cast<int4*>(out_q)[i] = quant4(reinterpret_cast<const float4*>(coeff)[i], c, qt, dz, dz32);
    else out_q[i] = quant1s(coeff[i], c, qt, dz, dz32);
  }
}

int run_quantize(gsnfs_ctx* ctx, cudaStream_t st, const float* d_coeff, uint32_t n, const gsnfs_counts* d_counts,
                 int channels, const float* qstep, const gsnfs_quant* quant, int32_t* d_qcoeff) {
  if (n == 0) return GSNFS_OK;
  QStepParams qs;
  for (int c = 0; c < GSNFS_MAX_CHANNELS; ++c) qs.step[c] = c < channels ? qstep[c] : 1.0f;
  const double dz = quant ? (double)quant->dz_round : (double)(1.0f / 3.0f);
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const bool vec4 = (channels % 4) == 0;
  const uint64_t tot = (uint64_t)n * (uint64_t)(vec4 ? channels / 4 : channels);
  const int grid = (int)min((uint64_t)ctx->num_sms * 8u, (tot + 255u) / 256u);     // 8 resident CTAs per SM, grid-stride
  GSNFS_KERNEL(ctx, st, "quantize");
  if (vec4) quantize_kernel<4><<<grid, 256, 0, st>>>(d_coeff, n, n_dev, channels, qs, dz, d_qcoeff);
  else quantize_kernel<1><<<grid, 256, 0, st>>>(d_coeff, n, n_dev, channels, qs, dz, d_qcoeff);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

// ------------------------------------------------------------------------------------------------
static size_t raht_smem_bytes(int C) {
  return sizeof(float) * (size_t)T * C + 2 * sizeof(TileMeta) + (sizeof(double) + sizeof(float)) * ((C + 3) & ~3);
}

int raht_setup(gsnfs_ctx* ctx) {
  // the attribute belongs to the function on the device, not to this context: always the library-wide maximum
  const size_t smem = raht_smem_bytes(GSNFS_MAX_CHANNELS);
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_forward_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_forward_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_inverse_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(raht_inverse_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  return GSNFS_OK;
}

template <typename K>
static int coop_grid(gsnfs_ctx* ctx, int slot, K kernel, size_t smem, uint32_t want, int* out, int threads = 256) {
  int per_sm = ctx->occ_cache[slot];
  if (per_sm == 0 || ctx->occ_cache_smem[slot] != smem) {
    GSNFS_CUDA_OK(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem));
    ctx->occ_cache[slot] = per_sm;
    ctx->occ_cache_smem[slot] = smem;
  }
  if (per_sm < 1) { snprintf(ctx->err, sizeof(ctx->err), "raht kernel does not fit on an SM"); return GSNFS_E_CUDA; }
  const uint32_t cap = (uint32_t)per_sm * (uint32_t)ctx->num_sms;
  *out = (int)max(1u, min(cap, want));
  return GSNFS_OK;
}

int run_raht(gsnfs_ctx* ctx, cudaStream_t st, bool inverse, const uint64_t* d_keys, const uint32_t* d_weights,
             uint32_t n_voxels, gsnfs_counts* d_counts, int depth, const float* d_in_f, const int32_t* d_in_q,
             int channels, const float* qstep, const gsnfs_quant* quant, int32_t* d_out_q, float* d_out_f,
             const uint32_t* d_perm, const uint32_t* d_vstart, uint32_t* d_weights_out) {
  (void)depth;
  if (n_voxels == 0) return GSNFS_OK;
  const uint32_t want = (n_voxels + T - 1) / T;
  SchedPools sp;
  sp.rec = ctx->raht_rec; sp.hdr = ctx->raht_hdr; sp.pend = reinterpret_cast<PendRec*>(ctx->raht_pend);
  sp.tile_pend = ctx->raht_tile_pend; sp.bsum = ctx->raht_bsum;
  sp.hdr_cap = (uint32_t)ctx->raht_hdr_cap; sp.bsum_cap = ctx->raht_bsum_cap; sp.pool_rows = (uint32_t)ctx->raht_pool_rows;
  const bool fused = d_perm != nullptr;
  sp.perm = d_perm; sp.vstart = d_vstart; sp.gsrc = ctx->raht_gsrc; sp.weights_out = d_weights_out;
  if (fused) d_weights = d_weights_out;        // the transform kernels read the run lengths the schedule writes
  GatherArgs ga;
  ga.gsrc = fused ? ctx->raht_gsrc : nullptr; ga.perm = d_perm; ga.vstart = d_vstart; ga.partial = ctx->merge_partial;
  if (d_keys) {                                  // NULL: the schedule of the previous call on this context is reused
    int rc = launch_raht_schedule(ctx, st, d_keys, d_weights, n_voxels, d_counts, sp);
    if (rc != GSNFS_OK) return rc;
    ctx->sched_n = n_voxels;
    ctx->sched_stream = (void*)st;
  }
  QStepParams qs;
  for (int c = 0; c < GSNFS_MAX_CHANNELS; ++c) qs.step[c] = (qstep && c < channels) ? qstep[c] : 1.0f;
  const double dz = quant ? (double)quant->dz_round : (double)(1.0f / 3.0f);
  const double bias = quant ? (double)quant->recon_bias : 0.0;
  const size_t smem = raht_smem_bytes(channels);
  const bool vec4 = (channels % 4) == 0;
  int grid = 0;
  if (!inverse) {
    int has_q = (qstep != nullptr && d_out_q != nullptr) ? 1 : 0;
    void* args[] = {(void*)&d_in_f, (void*)&d_weights, (void*)&ga, (void*)&ctx->raht_rows, (void*)&ctx->raht_rec, (void*)&ctx->raht_hdr,
                    (void*)&ctx->raht_plan, (void*)&channels, (void*)&qs, (void*)&has_q, (void*)&dz,
                    (void*)&d_out_q, (void*)&d_out_f};
    void* fn = vec4 ? (void*)raht_forward_kernel<4> : (void*)raht_forward_kernel<1>;
    int rc = vec4 ? coop_grid(ctx, 1, raht_forward_kernel<4>, smem, want, &grid, kXT) : coop_grid(ctx, 2, raht_forward_kernel<1>, smem, want, &grid, kXT);
    if (rc != GSNFS_OK) return rc;
    GSNFS_KERNEL(ctx, st, "raht_forward");
    GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(kXT), args, smem, st));
    GSNFS_LAUNCH_CHECK(ctx, st);
  } else {
    void* args[] = {(void*)&d_in_q, (void*)&d_in_f, (void*)&d_weights, (void*)&ctx->raht_rows, (void*)&ctx->raht_rec,
                    (void*)&ctx->raht_hdr, (void*)&ctx->raht_plan, (void*)&channels, (void*)&qs, (void*)&bias,
                    (void*)&d_out_f};
    void* fn = vec4 ? (void*)raht_inverse_kernel<4> : (void*)raht_inverse_kernel<1>;
    int rc = vec4 ? coop_grid(ctx, 3, raht_inverse_kernel<4>, smem, want, &grid, kXT) : coop_grid(ctx, 4, raht_inverse_kernel<1>, smem, want, &grid, kXT);
    if (rc != GSNFS_OK) return rc;
    GSNFS_KERNEL(ctx, st, "raht_inverse");
    GSNFS_CUDA_OK(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(kXT), args, smem, st));
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  return GSNFS_OK;
}

}  // namespace gsnfs
