// Duplicate-voxel merge as a segmented reduction: the attributes of the
// Gaussians that fall into one voxel are replaced by their arithmetic mean [O9]; weight = count.
// Rows are gathered through the sorted permutation; a voxel holding one Gaussian (the common case)
// is a straight 16-byte-vector row copy, so the kernel is a 2 x 4C bytes/voxel HBM stream.
#include <type_traits>

#include "merge_long.cuh"

namespace gsnfs {

// Pre-pass of the long runs (merge_long.cuh): one 16-lane group per chunk of sorted positions.  Without long runs (every
// frame of the timed configs) a chunk costs two binary searches.
template <int VEC>
__global__ void __launch_bounds__(256) merge_long_kernel(const float* __restrict__ attr, int C, const uint32_t* __restrict__ perm,
                                                         const uint32_t* __restrict__ vstart,
                                                         const gsnfs_counts* __restrict__ counts, uint32_t nchunks,
                                                         double* __restrict__ partial) {
  const uint32_t nv = counts->n_voxels;
  if (nv == 0) return;
  for (uint32_t chunk = blockIdx.x * 16 + threadIdx.y; chunk < nchunks; chunk += gridDim.x * 16)
    long_chunk_partials<VEC>(attr, C, perm, vstart, nv, chunk, partial, (int)threadIdx.x, 16);
}

// VEC = 4: channels % 4 == 0, rows moved as float4 (rows are then 16-byte aligned);  VEC = 1: any C.
// Layout: threadIdx.x = vector lane inside a row (16 lanes), threadIdx.y = row slot; each thread keeps
// ROWS independent rows in flight to cover the start -> perm -> row dependent-load chain.
template <int VEC, int ROWS>
__global__ void __launch_bounds__(256) merge_kernel(const float* __restrict__ attr, int C,
                                                    const uint32_t* __restrict__ perm,
                                                    const uint32_t* __restrict__ vstart,
                                                    const gsnfs_counts* __restrict__ counts,
                                                    const double* __restrict__ partial,
                                                    float* __restrict__ merged, uint32_t* __restrict__ weights) {
  using VecT = typename std::conditional<VEC == 4, float4, float>::type;
  const uint32_t nv = counts->n_voxels;
  const int cv = C / VEC;                       // vectors per row
  const int lane = threadIdx.x;                 // 0..15
  const uint32_t rows_per_block = 16 * ROWS;
  for (uint32_t r0 = blockIdx.x * rows_per_block; r0 < nv; r0 += gridDim.x * rows_per_block) {
    uint32_t s[ROWS], e[ROWS], g[ROWS];
#pragma unroll
    for (int k = 0; k < ROWS; ++k) {
      const uint32_t v = r0 + threadIdx.y + 16 * k;
      s[k] = v < nv ? vstart[v] : 0u;
      e[k] = v < nv ? vstart[v + 1] : 0u;
    }
#pragma unroll
    for (int k = 0; k < ROWS; ++k) g[k] = (e[k] > s[k]) ? perm[s[k]] : 0u;
    for (int c = lane; c < cv; c += 16) {
      VecT x[ROWS];
#pragma unroll
      for (int k = 0; k < ROWS; ++k)
        if (e[k] > s[k]) x[k] = reinterpret_cast<const VecT*>(attr + (size_t)g[k] * C)[c];
#pragma unroll
      for (int k = 0; k < ROWS; ++k) {
        const uint32_t v = r0 + threadIdx.y + 16 * k;
        if (e[k] <= s[k]) continue;
        const uint32_t cnt = e[k] - s[k];
        if (cnt >= kLongRun) {                   // long run: chunk partials left by merge_long_kernel, in chunk order
          double a[VEC];
          long_run_sum<VEC>(partial, C, s[k], e[k], c, a);
          const double inv = (double)cnt;
          if constexpr (VEC == 4) x[k] = make_float4((float)(a[0] / inv), (float)(a[1] / inv), (float)(a[2] / inv), (float)(a[3] / inv));
          else x[k] = (float)(a[0] / inv);
        } else if (cnt > 1) {                    // rare: fp64 accumulation in sorted order, then mean
          if constexpr (VEC == 4) {
            double a0 = x[k].x, a1 = x[k].y, a2 = x[k].z, a3 = x[k].w;
            uint32_t q = s[k] + 1;
            for (; q + 4 <= e[k]; q += 4) {          // four rows in flight; the sums stay in sorted order
              uint32_t g4[4];
              float4 y4[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) g4[u] = perm[q + u];
#pragma unroll
              for (int u = 0; u < 4; ++u) y4[u] = reinterpret_cast<const float4*>(attr + (size_t)g4[u] * C)[c];
#pragma unroll
              for (int u = 0; u < 4; ++u) { a0 += y4[u].x; a1 += y4[u].y; a2 += y4[u].z; a3 += y4[u].w; }
            }
            for (; q < e[k]; ++q) {
              const float4 y = reinterpret_cast<const float4*>(attr + (size_t)perm[q] * C)[c];
              a0 += y.x; a1 += y.y; a2 += y.z; a3 += y.w;
            }
            const double inv = (double)cnt;
            x[k] = make_float4((float)(a0 / inv), (float)(a1 / inv), (float)(a2 / inv), (float)(a3 / inv));
          } else {
            double a0 = x[k];
            for (uint32_t q = s[k] + 1; q < e[k]; ++q) a0 += attr[(size_t)perm[q] * C + c];
            x[k] = (float)(a0 / (double)cnt);
          }
        }
        reinterpret_cast<VecT*>(merged + (size_t)v * C)[c] = x[k];
      }
    }
    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < ROWS; ++k) {
        const uint32_t v = r0 + threadIdx.y + 16 * k;
        if (v < nv) weights[v] = e[k] - s[k];
      }
    }
  }
}

int run_voxel_merge(gsnfs_ctx* ctx, cudaStream_t st, const float* d_attr, int channels, uint32_t n,
                    const uint32_t* d_perm, const uint32_t* d_voxel_start, const gsnfs_counts* d_counts,
                    float* d_merged, uint32_t* d_weights) {
  if (n == 0) return GSNFS_OK;
  constexpr int ROWS = 4;
  const dim3 block(16, 16);
  const uint32_t blocks_needed = (n + 16 * ROWS - 1) / (16 * ROWS);
  const uint32_t gcap = (uint32_t)ctx->num_sms * 32u;
  const int grid = (int)(blocks_needed < gcap ? blocks_needed : gcap);
  const uint32_t nchunks = (n + kLongChunk - 1) / kLongChunk;
  const int lgrid = (int)min((nchunks + 15u) / 16u, (uint32_t)ctx->num_sms * 8u);
  GSNFS_KERNEL(ctx, st, "merge_long");
  if (channels % 4 == 0)
    merge_long_kernel<4><<<lgrid, block, 0, st>>>(d_attr, channels, d_perm, d_voxel_start, d_counts, nchunks, ctx->merge_partial);
  else
    merge_long_kernel<1><<<lgrid, block, 0, st>>>(d_attr, channels, d_perm, d_voxel_start, d_counts, nchunks, ctx->merge_partial);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "merge");
  if (channels % 4 == 0)
    merge_kernel<4, ROWS><<<grid, block, 0, st>>>(d_attr, channels, d_perm, d_voxel_start, d_counts, ctx->merge_partial, d_merged,
                                                  d_weights);
  else
    merge_kernel<1, ROWS><<<grid, block, 0, st>>>(d_attr, channels, d_perm, d_voxel_start, d_counts, ctx->merge_partial, d_merged,
                                                  d_weights);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

}  // namespace gsnfs
