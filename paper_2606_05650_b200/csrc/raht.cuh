// Shared between the RAHT schedule (raht_schedule.cu) and the transform kernels (raht.cu).
#pragma once
#include "common.cuh"

namespace gsnfs {

constexpr int kPendCap = 128;          // >= 2 * 3 * GSNFS_MAX_DEPTH + 1 pending entries per tile
struct __align__(16) PendRec { uint32_t klo, khi, vidx, w; };   // a node of the next phase: code, first voxel, weight

struct SchedPools {
  uint4* rec;            // (toff + tile) * kRahtTile + j: {k | l << 8 | depth bucket << 16, a, b, vidx}
  RahtTileHdr* hdr;      // toff + tile
  PendRec* pend;         // (toff + tile) * kPendCap + rank
  uint32_t* tile_pend;   // toff + tile
  uint32_t* bsum;        // boff + tile / 256
  uint32_t hdr_cap;
  uint32_t bsum_cap;
  uint32_t pool_rows;    // capacity of the pending-row pool used by the transform kernels
  // fused merge (gsnfs_merge_raht_forward): leaf weight = run length in the sorted permutation
  const uint32_t* perm;      // NULL unless fused
  const uint32_t* vstart;
  uint32_t* gsrc;            // out: index of the first Gaussian of every voxel
  uint32_t* weights_out;     // out: run lengths
};

// Enqueues the schedule ("prelude") kernel: all phases, one cooperative launch.
int launch_raht_schedule(gsnfs_ctx* ctx, cudaStream_t st, const uint64_t* d_keys, const uint32_t* d_weights,
                         uint32_t n_voxels, gsnfs_counts* d_counts, const SchedPools& sp);

}  // namespace gsnfs
