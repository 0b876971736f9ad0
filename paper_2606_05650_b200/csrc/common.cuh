// Internal definitions shared by the gsnfs CUDA translation units (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "gsnfs.h"

namespace gsnfs {

constexpr int kRahtTile = 256;       // entries per RAHT tile (rows staged in shared memory)
constexpr int kRahtMaxPhases = 34;   // >= worst-case number of tile phases
constexpr int kSortItems = 16;       // keys per thread in a onesweep tile
constexpr int kSortThreads = 256;
constexpr int kSortTile = kSortItems * kSortThreads;
constexpr int kSortMaxPasses = 8;    // ceil(63 / 8)
constexpr int kOctTile = 2048;       // sorted keys per octree-build tile
constexpr int kOctLevels = 24;       // >= GSNFS_MAX_DEPTH + 2
constexpr int kScanTile = 2048;

struct SortPlan {
  int passes;
  int shift[kSortMaxPasses];
  int bits[kSortMaxPasses];
};

// Per-tile header of the RAHT schedule (one per tile per phase).
struct __align__(16) RahtTileHdr {
  uint16_t lev_end[64];   // lev_end[s] = end (exclusive) of the s-th non-empty level's records, s < nseg
  uint32_t pendmask[8];   // bit k set: entry k of the tile stays pending after this phase
  uint32_t pend_off;      // exclusive prefix of pending counts over the phase's earlier tiles
  uint32_t npend;
  uint32_t nent;          // valid entries in the tile | nseg << 16
  uint32_t nmerge;
};
static_assert(sizeof(RahtTileHdr) == 176, "RahtTileHdr layout");

// Device-resident description of the phase structure (data dependent).
struct RahtPlan {
  uint32_t nphases;
  uint32_t overflow;                  // the schedule did not fit the scratch, or `invalid`: the transform kernels write nothing
  uint32_t invalid;                   // voxel codes not sorted and unique, or a zero leaf weight
  uint32_t has_long;                  // fused merge: some voxel holds >= kLongRun Gaussians (merge_long.cuh)
  uint32_t M[kRahtMaxPhases + 2];     // active entries of phase p (1-based); M[1] = N_v
  uint32_t poff[kRahtMaxPhases + 2];  // row offset of phase p (p >= 2) in the idx / pending-row pools
  uint32_t toff[kRahtMaxPhases + 2];  // tile-header offset of phase p (records start at toff * kRahtTile)
#ifdef GSNFS_TIMELINE                 // developer builds only: globaltimer (ns) stamps written by CTA 0
  unsigned long long t_stamp[64];
#endif
};

struct ProfRec {
  const char* name;
  cudaEvent_t a, b;
};

}  // namespace gsnfs

struct gsnfs_ctx {
  int device;
  int num_sms;
  uint64_t max_points;
  int max_channels;
  int max_depth;
  uint64_t launches;
  char err[256];

  // optional per-kernel timing (gsnfs_profile_start/stop): one event pair per launch
  int prof_on;
  int prof_n;
  int prof_cap;
  gsnfs::ProfRec* prof;

  char* pool;
  size_t pool_bytes;

  // sort + octree build
  void* keys_a;            // max_points x 8
  void* keys_b;            // max_points x 8
  uint32_t* pay_a;
  uint32_t* pay_b;
  uint32_t* hist;          // kSortMaxPasses x 256
  uint32_t* sort_group_hist;  // 2 x sort_groups_cap x 256 (digit counts summed per 32 tiles, double buffered by pass parity)
  uint32_t sort_groups_cap;
  uint32_t* sort_tile_hist;   // tiles x 256
  size_t sort_zero_bytes;     // hist + sort_group_hist are contiguous; cleared by one memset
  uint32_t* oct_hist;      // kOctLevels x oct_tiles (level-major)
  uint32_t* oct_base;      // kOctLevels x oct_tiles
  uint32_t* oct_meta;      // level sizes [kOctLevels] + level offsets [kOctLevels]
  uint32_t oct_tiles_cap;

  // generic scan scratch
  uint32_t* scan_sums;     // per-tile sums
  uint32_t scan_tiles_cap;

  // RAHT
  uint4* raht_pend;        // pending entries {code, first voxel, node weight}, tile strided (raht_hdr_cap x 128)
  uint32_t* raht_bsum;     // pending counts summed per 256 tiles
  uint32_t* raht_gsrc;     // fused merge: first Gaussian of every voxel
  double* merge_partial;   // long-run merge: 2 x ceil(max_points / 256) x max_channels chunk partial sums (merge_long.cuh)
  uint32_t raht_bsum_cap;
  uint4* raht_rec;         // merge records
  gsnfs::RahtTileHdr* raht_hdr;
  uint32_t* raht_tile_pend;
  gsnfs::RahtPlan* raht_plan;
  float* raht_rows;        // pending-row pool (phases >= 2)
  uint64_t raht_pool_rows; // capacity (rows) of raht_idx / raht_rows
  uint64_t sched_n;        // row count of the schedule currently held in raht_rec / raht_hdr / raht_plan (0 = none)
  void* sched_stream;      // the stream that schedule was built on (reuse is only ordered on the same stream)
  uint32_t* h_flags;       // host-mapped: [0] != 0 <=> a kernel of this context found its scratch too small
  uint32_t* d_flags;       // device alias of h_flags
  uint64_t raht_rec_cap;
  uint64_t raht_hdr_cap;
  float* qparams;          // 2 x max_channels doubles (inv step / step) stored as double
  int occ_cache[16];       // cached cudaOccupancyMaxActiveBlocksPerMultiprocessor results (0 = not yet queried)
  size_t occ_cache_smem[16];

  // colour decorrelation: per-CTA partial moments of the KLT fit
  double* color_partial;
  uint32_t color_parts_cap;

  // rANS (occupancy bytes): histogram, strided word scratch, block states and offsets
  uint32_t* rans_hist;
  uint16_t* rans_scratch;
  uint32_t* rans_states;
  uint64_t* rans_off;
  uint64_t rans_blocks_cap;

  // RLGR: bytes of every block row and of every 256 block rows (stream offsets without a scan pass)
  uint64_t* rlgr_rowsum;
  uint64_t* rlgr_supersum;
  uint64_t rlgr_rows_cap;
  uint64_t rlgr_off_cap;   // entries of a block header at the smallest block size (staging of the *_host_packed calls)

  // decode
  uint64_t* dec_kmid;      // Morton codes of the decoder's middle level (max_points + 1 entries)
  uint32_t* dec_parent;    // (parent stream index << 3 | child digit) of every breadth-first node: occ_cap + max_points + 2
  uint64_t occ_cap;

  // host-frame staging (allocated on first use)
  char* fpool;
  size_t fpool_bytes;
  float* f_xyz;
  float* f_attr;
  float* f_merged;
  int32_t* f_q;
  uint8_t* f_occ;
  uint32_t* f_levels;
  uint32_t* f_perm;
  uint64_t* f_vkeys;
  uint32_t* f_vstart;
  uint32_t* f_weights;
  uint32_t* f_vxyz;
  gsnfs_counts* f_counts;
  uint32_t* f_bits;        // RLGR block header
  gsnfs_rlgr_info* f_info;
  uint8_t* f_stream;       // RLGR block streams (aliases f_merged)
  uint64_t f_stream_cap;
  cudaStream_t copy_stream;   // the large H2D copies of the *_host_packed calls overlap the position coder
  cudaEvent_t ev_a, ev_b;
};

namespace gsnfs {

#define GSNFS_CUDA_OK(ctx, expr)                                                              \
  do {                                                                                        \
    cudaError_t e__ = (expr);                                                                 \
    if (e__ != cudaSuccess) {                                                                 \
      snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, #expr,     \
               cudaGetErrorString(e__));                                                      \
      return GSNFS_E_CUDA;                                                                    \
    }                                                                                         \
  } while (0)

// Bracket every kernel launch: GSNFS_KERNEL(ctx, st, "name") before, GSNFS_LAUNCH_CHECK(ctx, st) after.
#define GSNFS_KERNEL(ctx, st, kname)                                         \
  do {                                                                       \
    if ((ctx)->prof_on && (ctx)->prof_n < (ctx)->prof_cap) {                 \
      (ctx)->prof[(ctx)->prof_n].name = (kname);                             \
      cudaEventRecord((ctx)->prof[(ctx)->prof_n].a, (st));                   \
    }                                                                        \
  } while (0)

#define GSNFS_LAUNCH_CHECK(ctx, st)                                          \
  do {                                                                       \
    (ctx)->launches++;                                                       \
    if ((ctx)->prof_on && (ctx)->prof_n < (ctx)->prof_cap) {                 \
      cudaEventRecord((ctx)->prof[(ctx)->prof_n].b, (st));                   \
      (ctx)->prof_n++;                                                       \
    }                                                                        \
    GSNFS_CUDA_OK(ctx, cudaPeekAtLastError());                               \
  } while (0)

__device__ __forceinline__ int msb64(unsigned long long x) { return 63 - __clzll((long long)x); }
__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}
__device__ __forceinline__ unsigned lanemask_le() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_le;" : "=r"(m));
  return m;
}
#ifdef GSNFS_TIMELINE
__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
#define GSNFS_TSTAMP(plan, i) do { if (blockIdx.x == 0 && threadIdx.x == 0 && (i) < 64) (plan)->t_stamp[(i)] = globaltimer_ns(); } while (0)
#else
#define GSNFS_TSTAMP(plan, i) do { } while (0)
#endif
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_volatile_u32(uint32_t* p, uint32_t v) {
  asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Exclusive scan of one value per thread over a 256-thread block.  `total` (optional) gets the sum.
__device__ __forceinline__ uint32_t block_excl_scan_256(uint32_t v, uint32_t* s_warp /*>= 9*/, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) s_warp[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < 8 ? s_warp[lane] : 0;
    uint32_t winc = w;
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += t;
    }
    if (lane < 8) s_warp[lane] = winc - w;
    if (lane == 7) s_warp[8] = winc;
  }
  __syncthreads();
  uint32_t res = inc - v + s_warp[warp];
  if (total) *total = s_warp[8];
  __syncthreads();
  return res;
}

// ---- entry points of the stage drivers (one per .cu) -------------------------------------------
int run_octree_encode(gsnfs_ctx* ctx, cudaStream_t st, const float* d_xyz, uint32_t n, const double lo[3],
                      const double scale[3], int depth, uint8_t* d_occ, uint64_t occ_capacity,
                      uint32_t* d_level_sizes, uint32_t* d_perm, uint64_t* d_voxel_keys,
                      uint32_t* d_voxel_start, gsnfs_counts* d_counts);
int run_voxel_merge(gsnfs_ctx* ctx, cudaStream_t st, const float* d_attr, int channels, uint32_t n,
                    const uint32_t* d_perm, const uint32_t* d_voxel_start, const gsnfs_counts* d_counts,
                    float* d_merged, uint32_t* d_weights);
bool octree_header_ok(const uint32_t* level_sizes, int depth, uint64_t occ_bytes);
int run_octree_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_occ, uint64_t occ_bytes,
                      const uint32_t* level_sizes, int depth, uint32_t* d_voxel_xyz, uint64_t* d_voxel_keys,
                      gsnfs_counts* d_counts);
int run_raht(gsnfs_ctx* ctx, cudaStream_t st, bool inverse, const uint64_t* d_keys, const uint32_t* d_weights,
             uint32_t n_voxels, gsnfs_counts* d_counts, int depth, const float* d_in_f,
             const int32_t* d_in_q, int channels, const float* qstep, const gsnfs_quant* quant,
             int32_t* d_out_q, float* d_out_f, const uint32_t* d_perm = nullptr, const uint32_t* d_vstart = nullptr,
             uint32_t* d_weights_out = nullptr);
int run_quantize(gsnfs_ctx* ctx, cudaStream_t st, const float* d_coeff, uint32_t n, const gsnfs_counts* d_counts,
                 int channels, const float* qstep, const gsnfs_quant* quant, int32_t* d_qcoeff);
int run_rlgr_encode(gsnfs_ctx* ctx, cudaStream_t st, const int32_t* d_q, uint32_t n, const gsnfs_counts* d_counts,
                    int channels, uint32_t block, uint32_t* d_block_bits, uint8_t* d_stream, uint64_t capacity,
                    gsnfs_rlgr_info* d_info);
int run_rlgr_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_stream, uint64_t stream_bytes,
                    const uint32_t* d_block_bits, uint32_t n, int channels, uint32_t block, int32_t* d_q,
                    gsnfs_rlgr_info* d_info);
int run_rans_encode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_data, uint64_t n, const uint32_t* n_dev, uint16_t* d_freq,
                    uint16_t* d_nwords, uint8_t* d_payload, uint64_t capacity, gsnfs_rlgr_info* d_info);
int run_rans_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_payload, uint64_t payload_bytes, const uint16_t* d_freq,
                    const uint16_t* d_nwords, uint64_t n, uint8_t* d_out, gsnfs_rlgr_info* d_info);
int rans_setup(gsnfs_ctx* ctx);
int run_klt_fit(gsnfs_ctx* ctx, cudaStream_t st, const float* d_attr, uint32_t n, const gsnfs_counts* d_counts, int channels,
                float* d_klt);
int run_color_apply(gsnfs_ctx* ctx, cudaStream_t st, bool inverse, const float* d_in, uint32_t n, const gsnfs_counts* d_counts,
                    int channels, const float* d_klt, float* d_out);
int color_setup(gsnfs_ctx* ctx);
int raht_setup(gsnfs_ctx* ctx);   // occupancy queries + attributes, called from gsnfs_create

}  // namespace gsnfs
