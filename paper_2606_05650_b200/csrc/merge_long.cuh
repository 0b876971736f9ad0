// Duplicate-voxel merge, long runs (PAPER.md:L89, L152-154 [O9]).  A voxel's Gaussians are summed in fp64 in sorted
// order by ONE lane group, which is the right thing for the runs of a frame (1-30 Gaussians) and a cliff for a coarse
// grid (a run of 100 000 rows is a 100 000-step serial chain: 61 ms for a 1M-point cloud in 8 voxels).  Runs of at least
// kLongRun rows are therefore summed chunk-wise: the sorted positions are cut into chunks of kLongChunk; a pre-pass that
// is spread over the whole grid leaves, per chunk, the partial sum of the long run that covers the chunk's first
// position (slot A) and of the long run that starts inside it (slot B; there is at most one of each, a run that both
// starts and ends inside one chunk is not long); the voxel's sum is then slot (A or B)[first chunk] + A[next chunk] +
// ... in chunk order.  The order of the additions is fixed by the positions alone, so the result is deterministic and
// the same in gsnfs_voxel_merge and in gsnfs_merge_raht_forward (bit for bit); shorter runs keep the plain in-order sum.
#pragma once
#include "common.cuh"

namespace gsnfs {

constexpr uint32_t kLongChunk = 256;
constexpr uint32_t kLongRun = 256;     // >= kLongChunk: such a run covers some chunk's first position or crosses its end

// index of the voxel that holds sorted position p (largest v with vstart[v] <= p); nv >= 1
__device__ __forceinline__ uint32_t voxel_of_position(const uint32_t* __restrict__ vstart, uint32_t nv, uint32_t p) {
  uint32_t lo = 0, hi = nv - 1;
  while (lo < hi) {
    const uint32_t mid = (lo + hi + 1) >> 1;
    if (__ldg(vstart + mid) <= p) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// fp64 sum of the rows perm[a .. b) (vector c of every row), in position order, four rows in flight
template <int VEC>
__device__ __forceinline__ void sum_rows(const float* __restrict__ attr, int C, const uint32_t* __restrict__ perm, uint32_t a,
                                         uint32_t b, int c, double (&acc)[VEC]) {
  uint32_t q = a;
  if constexpr (VEC == 4) {
    for (; q + 4 <= b; q += 4) {
      uint32_t g4[4];
      float4 y4[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) g4[u] = perm[q + u];
#pragma unroll
      for (int u = 0; u < 4; ++u) y4[u] = reinterpret_cast<const float4*>(attr + (size_t)g4[u] * C)[c];
#pragma unroll
      for (int u = 0; u < 4; ++u) { acc[0] += y4[u].x; acc[1] += y4[u].y; acc[2] += y4[u].z; acc[3] += y4[u].w; }
    }
    for (; q < b; ++q) {
      const float4 y = reinterpret_cast<const float4*>(attr + (size_t)perm[q] * C)[c];
      acc[0] += y.x; acc[1] += y.y; acc[2] += y.z; acc[3] += y.w;
    }
  } else {
    for (; q < b; ++q) acc[0] += attr[(size_t)perm[q] * C + c];
  }
}

// Pre-pass body for one chunk, executed by a group of `lpr` lanes (lane l of the group takes vectors l, l + lpr, ...).
// partial: [2 * nchunks][C] doubles, slot A of chunk k at 2k, slot B at 2k + 1.
template <int VEC>
__device__ void long_chunk_partials(const float* __restrict__ attr, int C, const uint32_t* __restrict__ perm,
                                    const uint32_t* __restrict__ vstart, uint32_t nv, uint32_t chunk, double* __restrict__ partial,
                                    int l, int lpr) {
  const uint32_t n = __ldg(vstart + nv);
  const uint32_t p0 = chunk * kLongChunk;
  if (p0 >= n) return;
  const uint32_t p1 = min(p0 + kLongChunk, n);
  const int cv = C / VEC;
  const uint32_t v0 = voxel_of_position(vstart, nv, p0);
  const uint32_t e0 = __ldg(vstart + v0 + 1);
  if (e0 - __ldg(vstart + v0) >= kLongRun) {
    double* out = partial + (size_t)(2 * chunk) * C;
    for (int c = l; c < cv; c += lpr) {
      double acc[VEC] = {};
      sum_rows<VEC>(attr, C, perm, p0, min(e0, p1), c, acc);
#pragma unroll
      for (int u = 0; u < VEC; ++u) out[VEC * c + u] = acc[u];
    }
  }
  if (e0 < p1) {                                   // another voxel holds the chunk's last position
    const uint32_t v1 = voxel_of_position(vstart, nv, p1 - 1);
    const uint32_t s1 = __ldg(vstart + v1);
    if (__ldg(vstart + v1 + 1) - s1 >= kLongRun) {
      double* out = partial + (size_t)(2 * chunk + 1) * C;
      for (int c = l; c < cv; c += lpr) {
        double acc[VEC] = {};
        sum_rows<VEC>(attr, C, perm, s1, p1, c, acc);
#pragma unroll
        for (int u = 0; u < VEC; ++u) out[VEC * c + u] = acc[u];
      }
    }
  }
}

// Sum of the long run [s, e) from the chunk partials (vector c), in chunk order.
template <int VEC>
__device__ __forceinline__ void long_run_sum(const double* __restrict__ partial, int C, uint32_t s, uint32_t e, int c,
                                             double (&acc)[VEC]) {
  const uint32_t cf = s / kLongChunk, cl = (e - 1) / kLongChunk;
  const double* first = partial + (size_t)(2 * cf + ((s % kLongChunk) ? 1u : 0u)) * C + VEC * c;
#pragma unroll
  for (int u = 0; u < VEC; ++u) acc[u] = __ldcg(first + u);
  for (uint32_t k = cf + 1; k <= cl; ++k) {
    const double* pk = partial + (size_t)(2 * k) * C + VEC * c;
#pragma unroll
    for (int u = 0; u < VEC; ++u) acc[u] += __ldcg(pk + u);
  }
}

}  // namespace gsnfs
