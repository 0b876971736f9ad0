// C ABI of libgsnfs.so (see include/gsnfs.h): argument validation, context scratch, stage drivers.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "common.cuh"

namespace gsnfs {
int octree_encode_setup(gsnfs_ctx* ctx);

struct Bump {
  size_t off = 0;
  size_t take(size_t bytes) {
    const size_t o = off;
    off += (bytes + 255) & ~(size_t)255;
    return o;
  }
};
}  // namespace gsnfs

using namespace gsnfs;

namespace {
// Every entry point runs on the context's device and leaves the caller's current device as it found it.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  cudaError_t enter(int dev) {
    cudaError_t e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return e;
    if (prev != dev) { e = cudaSetDevice(dev); switched = (e == cudaSuccess); }
    return e;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
#define GSNFS_ON_DEVICE(ctx) DeviceGuard guard__; GSNFS_CUDA_OK(ctx, guard__.enter((ctx)->device))

// A scratch overflow is found on the device, after the call that caused it has returned: the kernel sets
// gsnfs_counts.status bit 1 (when the call was given a d_counts) and a host-mapped flag that the NEXT entry point
// on this context (or gsnfs_poll_status) reports once as GSNFS_E_CAPACITY.
int take_sticky(gsnfs_ctx* ctx) {
  if (ctx->h_flags && *(volatile uint32_t*)ctx->h_flags) {
    *(volatile uint32_t*)ctx->h_flags = 0;
    ctx->sched_n = 0;
    snprintf(ctx->err, sizeof(ctx->err), "an earlier RAHT call on this context overflowed its schedule scratch "
             "(unsorted or duplicate voxel keys?); its outputs were not written");
    return GSNFS_E_CAPACITY;
  }
  return GSNFS_OK;
}
bool quant_ok(const gsnfs_quant* q) {
  if (!q) return true;
  return isfinite(q->dz_round) && q->dz_round >= 0.f && q->dz_round <= 1.f && isfinite(q->recon_bias) &&
         q->recon_bias >= 0.f && q->recon_bias < 1.f;
}
}  // namespace

extern "C" {

const char* gsnfs_version(void) { return "gsnfs-b200 0.1 (sm_100a)"; }

const char* gsnfs_strerror(int status) {
  switch (status) {
    case GSNFS_OK: return "ok";
    case GSNFS_E_INVALID_ARGUMENT: return "invalid argument";
    case GSNFS_E_CAPACITY: return "capacity exceeded (context scratch or caller buffer too small)";
    case GSNFS_E_CUDA: return "CUDA error (see gsnfs_last_error)";
    case GSNFS_E_CORRUPT_STREAM: return "corrupt occupancy stream";
    case GSNFS_E_UNIMPLEMENTED: return "not implemented";
    default: return "unknown status";
  }
}

const char* gsnfs_last_error(const gsnfs_ctx* ctx) { return ctx ? ctx->err : "null context"; }
int gsnfs_poll_status(gsnfs_ctx* ctx) { return ctx ? take_sticky(ctx) : GSNFS_E_INVALID_ARGUMENT; }
uint64_t gsnfs_launch_count(const gsnfs_ctx* ctx) { return ctx ? ctx->launches : 0; }

uint64_t gsnfs_occ_capacity(uint64_t n, int depth) {
  if (depth < 1 || depth > GSNFS_MAX_DEPTH) return 0;
  uint64_t s = 0, pw = 1;
  for (int d = 0; d < depth; ++d) {
    s += pw < n ? pw : n;
    if (pw < (1ull << 62)) pw <<= 3;
  }
  return (s + 15) & ~15ull;
}

static int create_impl(gsnfs_ctx* c) {
  GSNFS_ON_DEVICE(c);
  GSNFS_CUDA_OK(c, cudaHostAlloc((void**)&c->h_flags, 64, cudaHostAllocMapped));
  memset(c->h_flags, 0, 64);
  GSNFS_CUDA_OK(c, cudaHostGetDevicePointer((void**)&c->d_flags, c->h_flags, 0));
  cudaDeviceProp prop;
  GSNFS_CUDA_OK(c, cudaGetDeviceProperties(&prop, c->device));
  c->num_sms = prop.multiProcessorCount;
  if (!prop.cooperativeLaunch) {
    snprintf(c->err, sizeof(c->err), "device lacks cooperative launch");
    return GSNFS_E_CUDA;
  }
  const uint64_t N = c->max_points;
  const int C = c->max_channels;
  const uint64_t stiles = N / 1024 + 2048;      // sort tiles hold 1024..kSortTile keys (balanced tiling)
  const uint64_t otiles = (N + kOctTile - 1) / kOctTile + 1;
  c->oct_tiles_cap = (uint32_t)otiles;
  c->occ_cap = gsnfs_occ_capacity(N, c->max_depth) + 16;
  c->scan_tiles_cap = (uint32_t)((c->occ_cap > N ? c->occ_cap : N) / kScanTile + 2);
  c->raht_pool_rows = N + 16384;          // sum of the phase sizes M_p, p >= 2
  c->raht_hdr_cap = 2 * N / kRahtTile + 4 * kRahtMaxPhases + 64;
  c->raht_rec_cap = c->raht_hdr_cap * kRahtTile;

  Bump b;
  const size_t o_keys_a = b.take(N * 8), o_keys_b = b.take(N * 8);
  const size_t o_pay_a = b.take(N * 4), o_pay_b = b.take(N * 4);
  const size_t o_hist = b.take((size_t)kSortMaxPasses * 256 * 4);
  c->sort_groups_cap = (uint32_t)(stiles / 32 + 2);
  const size_t o_sgrp = b.take((size_t)2 * c->sort_groups_cap * 256 * 4);
  const size_t o_zero_end = b.off;
  const size_t o_sth = b.take((size_t)stiles * 256 * 4);
  const size_t o_ohist = b.take((size_t)kOctLevels * otiles * 4), o_obase = b.take((size_t)kOctLevels * otiles * 4);
  const size_t o_ometa = b.take((size_t)2 * kOctLevels * 4);
  const size_t o_ssums = b.take((size_t)c->scan_tiles_cap * 4);
  c->raht_bsum_cap = (uint32_t)(c->raht_hdr_cap / 256 + 2 * kRahtMaxPhases + 8);
  const size_t o_rpend = b.take(c->raht_hdr_cap * 128 * sizeof(uint4));
  const size_t o_rbs = b.take((size_t)c->raht_bsum_cap * 4);
  const size_t o_rgs = b.take(N * 4);
  const size_t o_mpart = b.take(2 * (N / 256 + 2) * (size_t)C * 8);
  const size_t o_rrec = b.take(c->raht_rec_cap * sizeof(uint4));
  const size_t o_rhdr = b.take(c->raht_hdr_cap * sizeof(RahtTileHdr));
  const size_t o_rtp = b.take(c->raht_hdr_cap * 4);
  const size_t o_rplan = b.take(sizeof(RahtPlan));
  const size_t o_rrows = b.take(c->raht_pool_rows * (size_t)C * 4);
  c->rans_blocks_cap = c->occ_cap / GSNFS_RANS_BLOCK + 64;
  const size_t o_rah = b.take(256 * 4), o_ras = b.take(c->rans_blocks_cap * GSNFS_RANS_BLOCK * 2);
  const size_t o_rast = b.take(c->rans_blocks_cap * 4), o_rao = b.take((c->rans_blocks_cap + 1) * 8);
  c->color_parts_cap = (uint32_t)c->num_sms * 4u;
  const size_t o_colp = b.take((size_t)c->color_parts_cap * 3 * 135 * sizeof(double));
  c->rlgr_off_cap = (N / GSNFS_RLGR_MIN_BLOCK + 1) * (uint64_t)C + 1;
  c->rlgr_rows_cap = N / GSNFS_RLGR_MIN_BLOCK + 2;
  const size_t o_rlo = b.take(c->rlgr_rows_cap * 8), o_rls = b.take((c->rlgr_rows_cap / 256 + 2) * 8);
  const size_t o_dpar = b.take((c->occ_cap + N + 2) * 4), o_dkm = b.take((N + 1) * 8);
  c->pool_bytes = b.off;
  GSNFS_CUDA_OK(c, cudaMalloc((void**)&c->pool, c->pool_bytes));
  char* p = c->pool;
  c->keys_a = p + o_keys_a; c->keys_b = p + o_keys_b;
  c->pay_a = (uint32_t*)(p + o_pay_a); c->pay_b = (uint32_t*)(p + o_pay_b);
  c->hist = (uint32_t*)(p + o_hist); c->sort_group_hist = (uint32_t*)(p + o_sgrp); c->sort_tile_hist = (uint32_t*)(p + o_sth);
  c->sort_zero_bytes = o_zero_end - o_hist;
  c->oct_hist = (uint32_t*)(p + o_ohist); c->oct_base = (uint32_t*)(p + o_obase); c->oct_meta = (uint32_t*)(p + o_ometa);
  c->scan_sums = (uint32_t*)(p + o_ssums);
  c->raht_pend = (uint4*)(p + o_rpend); c->raht_bsum = (uint32_t*)(p + o_rbs);
  c->raht_rec = (uint4*)(p + o_rrec); c->raht_gsrc = (uint32_t*)(p + o_rgs);
  c->merge_partial = (double*)(p + o_mpart);
  c->raht_hdr = (RahtTileHdr*)(p + o_rhdr); c->raht_tile_pend = (uint32_t*)(p + o_rtp);
  c->raht_plan = (RahtPlan*)(p + o_rplan); c->raht_rows = (float*)(p + o_rrows);
  c->dec_parent = (uint32_t*)(p + o_dpar); c->dec_kmid = (uint64_t*)(p + o_dkm);
  c->rlgr_rowsum = (uint64_t*)(p + o_rlo); c->rlgr_supersum = (uint64_t*)(p + o_rls);
  c->color_partial = (double*)(p + o_colp);
  c->rans_hist = (uint32_t*)(p + o_rah); c->rans_scratch = (uint16_t*)(p + o_ras);
  c->rans_states = (uint32_t*)(p + o_rast); c->rans_off = (uint64_t*)(p + o_rao);
  GSNFS_CUDA_OK(c, cudaMemset(c->pool, 0, o_rrows));     // everything but the big row pool ...
  GSNFS_CUDA_OK(c, cudaMemset(p + o_dpar, 0, c->pool_bytes - o_dpar));   // ... and the decoder's parent / middle-level arrays
  int rc = octree_encode_setup(c);
  if (rc != GSNFS_OK) return rc;
  rc = color_setup(c);
  if (rc != GSNFS_OK) return rc;
  rc = rans_setup(c);
  if (rc != GSNFS_OK) return rc;
  return raht_setup(c);
}

int gsnfs_create(gsnfs_ctx** out, int device, uint64_t max_points, int max_channels, int max_depth) {
  if (!out) return GSNFS_E_INVALID_ARGUMENT;
  *out = nullptr;
  if (max_points == 0 || max_points >= (1ull << 30) || max_channels < 1 || max_channels > GSNFS_MAX_CHANNELS ||
      max_depth < 1 || max_depth > GSNFS_MAX_DEPTH)
    return GSNFS_E_INVALID_ARGUMENT;
  gsnfs_ctx* c = (gsnfs_ctx*)calloc(1, sizeof(gsnfs_ctx));
  if (!c) return GSNFS_E_CAPACITY;
  c->device = device;
  c->max_points = max_points;
  c->max_channels = max_channels;
  c->max_depth = max_depth;
  const int rc = create_impl(c);
  if (rc != GSNFS_OK) {
    fprintf(stderr, "gsnfs_create failed: %s\n", c->err);
    if (c->pool) cudaFree(c->pool);
    if (c->h_flags) cudaFreeHost(c->h_flags);
    free(c);
    return rc;
  }
  *out = c;
  return GSNFS_OK;
}

void gsnfs_destroy(gsnfs_ctx* ctx) {
  if (!ctx) return;
  DeviceGuard guard;
  guard.enter(ctx->device);
  if (ctx->h_flags) cudaFreeHost(ctx->h_flags);
  for (int i = 0; i < ctx->prof_cap; ++i) { cudaEventDestroy(ctx->prof[i].a); cudaEventDestroy(ctx->prof[i].b); }
  free(ctx->prof);
  if (ctx->pool) cudaFree(ctx->pool);
  if (ctx->fpool) {
    cudaFree(ctx->fpool);
    cudaStreamDestroy(ctx->copy_stream);
    cudaEventDestroy(ctx->ev_a);
    cudaEventDestroy(ctx->ev_b);
  }
  free(ctx);
}

#ifdef GSNFS_TIMELINE
int gsnfs_debug_read_plan(gsnfs_ctx* ctx, void* h_out, uint64_t bytes) {   // developer builds only; not in gsnfs.h
  if (!ctx || !h_out) return GSNFS_E_INVALID_ARGUMENT;
  if (bytes > sizeof(RahtPlan)) bytes = sizeof(RahtPlan);
  GSNFS_ON_DEVICE(ctx);
  GSNFS_CUDA_OK(ctx, cudaDeviceSynchronize());
  GSNFS_CUDA_OK(ctx, cudaMemcpy(h_out, ctx->raht_plan, bytes, cudaMemcpyDeviceToHost));
  return GSNFS_OK;
}
#endif

int gsnfs_profile_start(gsnfs_ctx* ctx, int max_records) {
  if (!ctx || max_records < 1) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  if (max_records > ctx->prof_cap) {
    ProfRec* np = (ProfRec*)realloc(ctx->prof, sizeof(ProfRec) * (size_t)max_records);
    if (!np) return GSNFS_E_CAPACITY;
    ctx->prof = np;
    for (int i = ctx->prof_cap; i < max_records; ++i) {
      GSNFS_CUDA_OK(ctx, cudaEventCreate(&ctx->prof[i].a));
      GSNFS_CUDA_OK(ctx, cudaEventCreate(&ctx->prof[i].b));
      ctx->prof_cap = i + 1;
    }
  }
  ctx->prof_n = 0;
  ctx->prof_on = 1;
  return GSNFS_OK;
}

int gsnfs_profile_stop(gsnfs_ctx* ctx, char* out, uint64_t out_cap) {
  if (!ctx || !out || out_cap < 2) return GSNFS_E_INVALID_ARGUMENT;
  ctx->prof_on = 0;
  GSNFS_ON_DEVICE(ctx);
  GSNFS_CUDA_OK(ctx, cudaDeviceSynchronize());
  // aggregate by kernel name (names are string literals; compare by content)
  struct Agg { const char* name; int count; double ms; };
  Agg agg[64];
  int na = 0;
  for (int i = 0; i < ctx->prof_n; ++i) {
    float ms = 0.f;
    GSNFS_CUDA_OK(ctx, cudaEventElapsedTime(&ms, ctx->prof[i].a, ctx->prof[i].b));
    int k = 0;
    for (; k < na; ++k) if (strcmp(agg[k].name, ctx->prof[i].name) == 0) break;
    if (k == na) { if (na == 64) continue; agg[na].name = ctx->prof[i].name; agg[na].count = 0; agg[na].ms = 0.0; ++na; }
    agg[k].count++;
    agg[k].ms += ms;
  }
  size_t off = 0;
  out[0] = 0;
  for (int k = 0; k < na; ++k) {
    const int w = snprintf(out + off, (size_t)out_cap - off, "%s %d %.6f\n", agg[k].name, agg[k].count, agg[k].ms);
    if (w < 0 || (size_t)w >= (size_t)out_cap - off) return GSNFS_E_CAPACITY;
    off += (size_t)w;
  }
  return GSNFS_OK;
}

int gsnfs_octree_encode(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_xyz, uint64_t n, const float bbox_min[3],
                        const float bbox_max[3], int depth, uint8_t* d_occ, uint64_t occ_capacity,
                        uint32_t* d_level_sizes, uint32_t* d_perm, uint64_t* d_voxel_keys, uint32_t* d_voxel_start,
                        gsnfs_counts* d_counts) {
  if (!ctx || !bbox_min || !bbox_max || !d_occ || !d_level_sizes || !d_voxel_start || !d_counts ||
      (n && (!d_xyz || !d_perm || !d_voxel_keys)))
    return GSNFS_E_INVALID_ARGUMENT;
  if (depth < 1 || depth > GSNFS_MAX_DEPTH || n >= (1ull << 30)) return GSNFS_E_INVALID_ARGUMENT;
  double lo[3], scale[3];
  for (int a = 0; a < 3; ++a) {
    const double l = (double)bbox_min[a], h = (double)bbox_max[a];
    if (!(h > l) || !isfinite(l) || !isfinite(h)) return GSNFS_E_INVALID_ARGUMENT;
    lo[a] = l;
    scale[a] = ldexp(1.0, depth) / (h - l);          // [O2] computed once on the host in fp64
  }
  if (n > ctx->max_points || depth > ctx->max_depth) return GSNFS_E_CAPACITY;
  if (occ_capacity < gsnfs_occ_capacity(n, depth) || (occ_capacity & 3)) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  return run_octree_encode(ctx, (cudaStream_t)stream, d_xyz, (uint32_t)n, lo, scale, depth, d_occ, occ_capacity,
                           d_level_sizes, d_perm, d_voxel_keys, d_voxel_start, d_counts);
}

int gsnfs_voxel_merge(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_attr, int channels, uint64_t n,
                      const uint32_t* d_perm, const uint32_t* d_voxel_start, const gsnfs_counts* d_counts,
                      float* d_merged, uint32_t* d_weights) {
  if (!ctx || !d_voxel_start || !d_counts || (n && (!d_attr || !d_perm || !d_merged || !d_weights)))
    return GSNFS_E_INVALID_ARGUMENT;
  if (channels < 1 || channels > GSNFS_MAX_CHANNELS || n >= (1ull << 30)) return GSNFS_E_INVALID_ARGUMENT;
  if (n > ctx->max_points) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  return run_voxel_merge(ctx, (cudaStream_t)stream, d_attr, channels, (uint32_t)n, d_perm, d_voxel_start, d_counts,
                         d_merged, d_weights);
}

int gsnfs_octree_decode(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* d_occ, uint64_t occ_bytes,
                        const uint32_t* level_sizes, int depth, uint32_t* d_voxel_xyz, uint64_t* d_voxel_keys,
                        gsnfs_counts* d_counts) {
  if (!ctx || !level_sizes || !d_counts) return GSNFS_E_INVALID_ARGUMENT;
  if (depth < 1 || depth > GSNFS_MAX_DEPTH) return GSNFS_E_INVALID_ARGUMENT;
  if (level_sizes[depth] && (!d_occ || !d_voxel_xyz)) return GSNFS_E_INVALID_ARGUMENT;
  if (depth > ctx->max_depth) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  return run_octree_decode(ctx, (cudaStream_t)stream, d_occ, occ_bytes, level_sizes, depth, d_voxel_xyz, d_voxel_keys,
                           d_counts);
}

static int raht_check(gsnfs_ctx* ctx, gsnfs_stream stream, const uint64_t* keys, bool keys_required, uint64_t n, int depth,
                      int channels, const float* qstep, const gsnfs_quant* quant) {
  if (!ctx) return GSNFS_E_INVALID_ARGUMENT;
  int rc = take_sticky(ctx);
  if (rc != GSNFS_OK) return rc;
  if (depth < 1 || depth > GSNFS_MAX_DEPTH || channels < 1 || channels > GSNFS_MAX_CHANNELS || n >= (1ull << 30))
    return GSNFS_E_INVALID_ARGUMENT;
  if (n && !keys) {
    // schedule reuse: only where the header allows it, only a schedule of n rows built on this very stream
    if (keys_required || ctx->sched_n != n || ctx->sched_stream != (void*)stream) return GSNFS_E_INVALID_ARGUMENT;
  }
  if (!quant_ok(quant)) return GSNFS_E_INVALID_ARGUMENT;
  if (qstep)
    for (int c = 0; c < channels; ++c)
      if (!(qstep[c] > 0.f) || !isfinite(qstep[c])) return GSNFS_E_INVALID_ARGUMENT;
  if (n > ctx->max_points || channels > ctx->max_channels) return GSNFS_E_CAPACITY;
  return GSNFS_OK;
}

// a failed RAHT call leaves no schedule behind to reuse
static int raht_done(gsnfs_ctx* ctx, int rc) {
  if (rc != GSNFS_OK) ctx->sched_n = 0;
  return rc;
}

int gsnfs_raht_forward(gsnfs_ctx* ctx, gsnfs_stream stream, const uint64_t* d_voxel_keys, const uint32_t* d_weights,
                       uint64_t n_voxels, gsnfs_counts* d_counts, int depth, const float* d_attr, int channels,
                       const float* qstep, const gsnfs_quant* quant, int32_t* d_qcoeff, float* d_coeff) {
  int rc = raht_check(ctx, stream, d_voxel_keys, false, n_voxels, depth, channels, qstep, quant);
  if (rc != GSNFS_OK) return rc;
  if (n_voxels && (!d_attr || (!d_qcoeff && !d_coeff) || (d_qcoeff && !qstep))) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  return raht_done(ctx, run_raht(ctx, (cudaStream_t)stream, false, d_voxel_keys, d_weights, (uint32_t)n_voxels, d_counts, depth,
                                 d_attr, nullptr, channels, qstep, quant, d_qcoeff, d_coeff));
}

int gsnfs_merge_raht_forward(gsnfs_ctx* ctx, gsnfs_stream stream, const uint64_t* d_voxel_keys, const uint32_t* d_perm,
                             const uint32_t* d_voxel_start, uint64_t n, gsnfs_counts* d_counts, int depth,
                             const float* d_attr, int channels, const float* qstep, const gsnfs_quant* quant,
                             uint32_t* d_weights_out, int32_t* d_qcoeff, float* d_coeff) {
  int rc = raht_check(ctx, stream, d_voxel_keys, true, n, depth, channels, qstep, quant);
  if (rc != GSNFS_OK) return rc;
  if (!d_counts || (n && (!d_perm || !d_voxel_start || !d_attr || !d_weights_out || (!d_qcoeff && !d_coeff) || (d_qcoeff && !qstep))))
    return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  return raht_done(ctx, run_raht(ctx, (cudaStream_t)stream, false, d_voxel_keys, nullptr, (uint32_t)n, d_counts, depth, d_attr,
                                 nullptr, channels, qstep, quant, d_qcoeff, d_coeff, d_perm, d_voxel_start, d_weights_out));
}

int gsnfs_quantize(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_coeff, uint64_t n_rows,
                   const gsnfs_counts* d_counts, int channels, const float* qstep, const gsnfs_quant* quant,
                   int32_t* d_qcoeff) {
  if (!ctx || !qstep || (n_rows && (!d_coeff || !d_qcoeff))) return GSNFS_E_INVALID_ARGUMENT;
  if (channels < 1 || channels > GSNFS_MAX_CHANNELS || n_rows >= (1ull << 30) || !quant_ok(quant)) return GSNFS_E_INVALID_ARGUMENT;
  for (int c = 0; c < channels; ++c)
    if (!(qstep[c] > 0.f) || !isfinite(qstep[c])) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  return run_quantize(ctx, (cudaStream_t)stream, d_coeff, (uint32_t)n_rows, d_counts, channels, qstep, quant, d_qcoeff);
}

int gsnfs_raht_inverse(gsnfs_ctx* ctx, gsnfs_stream stream, const uint64_t* d_voxel_keys, const uint32_t* d_weights,
                       uint64_t n_voxels, gsnfs_counts* d_counts, int depth, const int32_t* d_qcoeff,
                       const float* d_coeff, int channels, const float* qstep, const gsnfs_quant* quant,
                       float* d_attr_out) {
  int rc = raht_check(ctx, stream, d_voxel_keys, false, n_voxels, depth, channels, qstep, quant);
  if (rc != GSNFS_OK) return rc;
  if (n_voxels && (!d_attr_out || (!d_qcoeff && !d_coeff) || (d_qcoeff && !qstep))) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  return raht_done(ctx, run_raht(ctx, (cudaStream_t)stream, true, d_voxel_keys, d_weights, (uint32_t)n_voxels, d_counts, depth,
                                 d_coeff, d_qcoeff, channels, d_qcoeff ? qstep : nullptr, quant, nullptr, d_attr_out));
}

// ---- colour decorrelation in front of RAHT -----------------------------------------------------------
static bool color_channels_ok(int channels) { return channels >= 11 && (channels - 11) % 3 == 0 && (channels - 11) / 3 <= 15; }

uint64_t gsnfs_klt_floats(int channels) {
  if (!color_channels_ok(channels)) return 0;
  const uint64_t K = (uint64_t)(channels - 11) / 3;
  return 3 * (2 * K + K * K);
}

int gsnfs_klt_fit(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_attr, uint64_t n_rows, const gsnfs_counts* d_counts,
                  int channels, float* d_klt) {
  if (!ctx || !color_channels_ok(channels) || n_rows >= (1ull << 30)) return GSNFS_E_INVALID_ARGUMENT;
  if (channels > 11 && (!d_klt || (n_rows && !d_attr))) return GSNFS_E_INVALID_ARGUMENT;
  if (n_rows > ctx->max_points || channels > GSNFS_MAX_CHANNELS) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  return run_klt_fit(ctx, (cudaStream_t)stream, d_attr, (uint32_t)n_rows, d_counts, channels, d_klt);
}

static int color_apply(gsnfs_ctx* ctx, gsnfs_stream stream, bool inverse, const float* d_in, uint64_t n_rows,
                       const gsnfs_counts* d_counts, int channels, const float* d_klt, float* d_out) {
  if (!ctx || !color_channels_ok(channels) || n_rows >= (1ull << 30) || (n_rows && (!d_in || !d_out)))
    return GSNFS_E_INVALID_ARGUMENT;
  if (n_rows > ctx->max_points) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  return run_color_apply(ctx, (cudaStream_t)stream, inverse, d_in, (uint32_t)n_rows, d_counts, channels, d_klt, d_out);
}

int gsnfs_color_forward(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_attr, uint64_t n_rows,
                        const gsnfs_counts* d_counts, int channels, const float* d_klt, float* d_out) {
  return color_apply(ctx, stream, false, d_attr, n_rows, d_counts, channels, d_klt, d_out);
}

int gsnfs_color_inverse(gsnfs_ctx* ctx, gsnfs_stream stream, const float* d_attr, uint64_t n_rows,
                        const gsnfs_counts* d_counts, int channels, const float* d_klt, float* d_out) {
  return color_apply(ctx, stream, true, d_attr, n_rows, d_counts, channels, d_klt, d_out);
}

// ---- RLGR entropy coder for the quantised coefficients ----------------------------------------------
uint64_t gsnfs_rlgr_blocks(uint64_t n_rows, int channels, int block_size) {
  if (block_size < GSNFS_RLGR_MIN_BLOCK || block_size > GSNFS_RLGR_MAX_BLOCK || channels < 1) return 0;
  return ((n_rows + (uint64_t)block_size - 1) / (uint64_t)block_size) * (uint64_t)channels;
}

uint64_t gsnfs_rlgr_capacity(uint64_t n_rows, int channels, int block_size) {
  const uint64_t nb = gsnfs_rlgr_blocks(n_rows, channels, block_size);
  return nb ? n_rows * (uint64_t)channels * 4ull + nb * 4ull : 0;
}

int gsnfs_rlgr_encode(gsnfs_ctx* ctx, gsnfs_stream stream, const int32_t* d_qcoeff, uint64_t n_rows,
                      const gsnfs_counts* d_counts, int channels, int block_size, uint32_t* d_block_bits,
                      uint8_t* d_stream, uint64_t stream_capacity, gsnfs_rlgr_info* d_info) {
  if (!ctx || !d_info || (n_rows && (!d_qcoeff || !d_block_bits || !d_stream))) return GSNFS_E_INVALID_ARGUMENT;
  if (channels < 1 || channels > GSNFS_MAX_CHANNELS || n_rows >= (1ull << 30) || block_size < GSNFS_RLGR_MIN_BLOCK ||
      block_size > GSNFS_RLGR_MAX_BLOCK || ((uintptr_t)d_stream & 3))
    return GSNFS_E_INVALID_ARGUMENT;
  if (n_rows > ctx->max_points || channels > ctx->max_channels) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  return run_rlgr_encode(ctx, (cudaStream_t)stream, d_qcoeff, (uint32_t)n_rows, d_counts, channels, (uint32_t)block_size,
                         d_block_bits, d_stream, stream_capacity, d_info);
}

int gsnfs_rlgr_decode(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* d_stream, uint64_t stream_bytes,
                      const uint32_t* d_block_bits, uint64_t n_rows, int channels, int block_size, int32_t* d_qcoeff,
                      gsnfs_rlgr_info* d_info) {
  if (!ctx || !d_info || (n_rows && (!d_qcoeff || !d_block_bits || (!d_stream && stream_bytes)))) return GSNFS_E_INVALID_ARGUMENT;
  if (channels < 1 || channels > GSNFS_MAX_CHANNELS || n_rows >= (1ull << 30) || block_size < GSNFS_RLGR_MIN_BLOCK ||
      block_size > GSNFS_RLGR_MAX_BLOCK || ((uintptr_t)d_stream & 3))
    return GSNFS_E_INVALID_ARGUMENT;
  if (n_rows > ctx->max_points || channels > ctx->max_channels) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  return run_rlgr_decode(ctx, (cudaStream_t)stream, d_stream, stream_bytes, d_block_bits, (uint32_t)n_rows, channels,
                         (uint32_t)block_size, d_qcoeff, d_info);
}

// ---- rANS entropy coder for the occupancy bytes -------------------------------------------------------
uint64_t gsnfs_rans_blocks(uint64_t n) { return (n + GSNFS_RANS_BLOCK - 1) / GSNFS_RANS_BLOCK; }
uint64_t gsnfs_rans_capacity(uint64_t n) { return n + n / 2 + 4 * gsnfs_rans_blocks(n) + 16; }     // 12 bits per byte at worst

int gsnfs_rans_encode(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* d_data, uint64_t n, const gsnfs_counts* d_counts,
                      uint16_t* d_freq, uint16_t* d_nwords, uint8_t* d_payload, uint64_t payload_capacity,
                      gsnfs_rans_info* d_info) {
  if (!ctx || !d_freq || !d_info || (n && (!d_data || !d_nwords || !d_payload)) || ((uintptr_t)d_data & 3))
    return GSNFS_E_INVALID_ARGUMENT;
  if (n >= (1ull << 32)) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  return run_rans_encode(ctx, (cudaStream_t)stream, d_data, n, d_counts ? &d_counts->occ_bytes : nullptr, d_freq, d_nwords,
                         d_payload, payload_capacity, d_info);
}

int gsnfs_rans_decode(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* d_payload, uint64_t payload_bytes,
                      const uint16_t* d_freq, const uint16_t* d_nwords, uint64_t n, uint8_t* d_out, gsnfs_rans_info* d_info) {
  if (!ctx || !d_freq || !d_info || (n && (!d_payload || !d_nwords || !d_out))) return GSNFS_E_INVALID_ARGUMENT;
  if (n >= (1ull << 32)) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  return run_rans_decode(ctx, (cudaStream_t)stream, d_payload, payload_bytes, d_freq, d_nwords, n, d_out, d_info);
}

// ---- whole-frame calls on host buffers -----------------------------------------------------------
static int frame_pool(gsnfs_ctx* c) {
  if (c->fpool) return GSNFS_OK;
  const uint64_t N = c->max_points;
  const size_t C = (size_t)c->max_channels;
  Bump b;
  const size_t o_xyz = b.take(N * 12), o_attr = b.take(N * C * 4), o_mrg = b.take(N * C * 4), o_q = b.take(N * C * 4);
  const size_t o_occ = b.take(c->occ_cap), o_lev = b.take(256), o_perm = b.take(N * 4), o_vk = b.take(N * 8);
  const size_t o_vs = b.take((N + 1) * 4), o_w = b.take(N * 4), o_vx = b.take(N * 12), o_cnt = b.take(256);
  const size_t o_bits = b.take(c->rlgr_off_cap * 4), o_info = b.take(256);
  // create everything first and publish it last: a context whose pool, copy stream or events could not be created keeps
  // fpool == NULL, so the next call tries again instead of running on a null stream
  char* p = nullptr;
  cudaStream_t cs = nullptr;
  cudaEvent_t ea = nullptr, eb = nullptr;
  cudaError_t e = cudaMalloc((void**)&p, b.off);
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ea, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&eb, cudaEventDisableTiming);
  if (e != cudaSuccess) {
    if (eb) cudaEventDestroy(eb);
    if (ea) cudaEventDestroy(ea);
    if (cs) cudaStreamDestroy(cs);
    if (p) cudaFree(p);
    snprintf(c->err, sizeof(c->err), "host-frame staging (%zu bytes, copy stream, events): %s", b.off, cudaGetErrorString(e));
    return GSNFS_E_CUDA;
  }
  c->fpool_bytes = b.off;
  c->f_xyz = (float*)(p + o_xyz); c->f_attr = (float*)(p + o_attr); c->f_merged = (float*)(p + o_mrg);
  c->f_q = (int32_t*)(p + o_q); c->f_occ = (uint8_t*)(p + o_occ); c->f_levels = (uint32_t*)(p + o_lev);
  c->f_perm = (uint32_t*)(p + o_perm); c->f_vkeys = (uint64_t*)(p + o_vk); c->f_vstart = (uint32_t*)(p + o_vs);
  c->f_weights = (uint32_t*)(p + o_w); c->f_vxyz = (uint32_t*)(p + o_vx); c->f_counts = (gsnfs_counts*)(p + o_cnt);
  c->f_bits = (uint32_t*)(p + o_bits); c->f_info = (gsnfs_rlgr_info*)(p + o_info);
  c->f_stream = (uint8_t*)c->f_merged;                 // the fused encoder never materialises the merged tensor
  c->f_stream_cap = N * C * 4;
  c->copy_stream = cs; c->ev_a = ea; c->ev_b = eb;
  c->fpool = p;
  return GSNFS_OK;
}

static int frame_encode_host_impl(gsnfs_ctx* ctx, gsnfs_stream stream, const float* h_xyz, const float* h_attr, uint64_t n,
                            int channels, const float bbox_min[3], const float bbox_max[3], int depth,
                            const float* qstep, const gsnfs_quant* quant, uint8_t* h_occ, uint64_t occ_capacity,
                            uint32_t* h_level_sizes, uint32_t* h_weights, int32_t* h_qcoeff, gsnfs_counts* h_counts) {
  if (!ctx || !h_occ || !h_level_sizes || !h_counts || !qstep || (n && (!h_xyz || !h_attr || !h_weights || !h_qcoeff)))
    return GSNFS_E_INVALID_ARGUMENT;
  if (n > ctx->max_points || channels > ctx->max_channels || channels < 1) return GSNFS_E_CAPACITY;
  GSNFS_ON_DEVICE(ctx);
  int rc = frame_pool(ctx);
  if (rc != GSNFS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const uint64_t cap = gsnfs_occ_capacity(n, depth);
  if (cap == 0 || occ_capacity < cap || cap > ctx->occ_cap) return depth < 1 || depth > GSNFS_MAX_DEPTH ? GSNFS_E_INVALID_ARGUMENT : GSNFS_E_CAPACITY;
  const size_t C = (size_t)channels;
  if (n) {
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_xyz, h_xyz, n * 12, cudaMemcpyHostToDevice, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_attr, h_attr, n * C * 4, cudaMemcpyHostToDevice, st));
  }
  rc = gsnfs_octree_encode(ctx, stream, ctx->f_xyz, n, bbox_min, bbox_max, depth, ctx->f_occ, cap, ctx->f_levels,
                           ctx->f_perm, ctx->f_vkeys, ctx->f_vstart, ctx->f_counts);
  if (rc != GSNFS_OK) return rc;
  rc = gsnfs_merge_raht_forward(ctx, stream, ctx->f_vkeys, ctx->f_perm, ctx->f_vstart, n, ctx->f_counts, depth, ctx->f_attr,
                                channels, qstep, quant, ctx->f_weights, ctx->f_q, nullptr);
  if (rc != GSNFS_OK) return rc;
  // header first: the sizes of the remaining copies depend on it
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_counts, ctx->f_counts, sizeof(gsnfs_counts), cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_level_sizes, ctx->f_levels, sizeof(uint32_t) * (depth + 1), cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaStreamSynchronize(st));
  const uint64_t nv = h_counts->n_voxels, ob = h_counts->occ_bytes;
  if (nv) {
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_occ, ctx->f_occ, ob, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_weights, ctx->f_weights, nv * 4, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_qcoeff, ctx->f_q, nv * C * 4, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaStreamSynchronize(st));
  }
  return GSNFS_OK;
}

static int frame_decode_host_impl(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* h_occ, uint64_t occ_bytes,
                            const uint32_t* level_sizes, int depth, const uint32_t* h_weights, const int32_t* h_qcoeff,
                            int channels, const float* qstep, const gsnfs_quant* quant, uint32_t* h_voxel_xyz,
                            float* h_attr, gsnfs_counts* h_counts) {
  if (!ctx || !level_sizes || !h_counts || !qstep) return GSNFS_E_INVALID_ARGUMENT;
  if (depth < 1 || depth > GSNFS_MAX_DEPTH) return GSNFS_E_INVALID_ARGUMENT;
  const uint64_t nv = level_sizes[depth];
  if (nv && (!h_occ || !h_qcoeff || !h_voxel_xyz || !h_attr)) return GSNFS_E_INVALID_ARGUMENT;
  if (nv > ctx->max_points || channels > ctx->max_channels || channels < 1 || occ_bytes + 1 > ctx->occ_cap)
    return GSNFS_E_CAPACITY;
  // header checks that need no device [O12]: an inconsistent header is reported before a byte is copied
  if (!octree_header_ok(level_sizes, depth, occ_bytes)) {
    h_counts->n_voxels = 0; h_counts->occ_bytes = (uint32_t)occ_bytes; h_counts->status = 1; h_counts->reserved = 0;
    return GSNFS_OK;
  }
  if (h_weights)
    for (uint64_t i = 0; i < nv; ++i)
      if (h_weights[i] == 0) return GSNFS_E_INVALID_ARGUMENT;                // a leaf of weight 0 has no transform [R1]
  GSNFS_ON_DEVICE(ctx);
  int rc = frame_pool(ctx);
  if (rc != GSNFS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t C = (size_t)channels;
  if (nv) {
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_occ, h_occ, occ_bytes, cudaMemcpyHostToDevice, st));
    if (h_weights) GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_weights, h_weights, nv * 4, cudaMemcpyHostToDevice, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_q, h_qcoeff, nv * C * 4, cudaMemcpyHostToDevice, st));
  }
  rc = gsnfs_octree_decode(ctx, stream, ctx->f_occ, occ_bytes, level_sizes, depth, ctx->f_vxyz, ctx->f_vkeys, ctx->f_counts);
  if (rc != GSNFS_OK) return rc;
  // f_counts chains the decoder's verdict on the device: a stream found corrupt there leaves N_v = 0, and the
  // inverse transform is then a no-op instead of a walk over stale codes
  rc = gsnfs_raht_inverse(ctx, stream, ctx->f_vkeys, h_weights ? ctx->f_weights : nullptr, nv, ctx->f_counts, depth, ctx->f_q,
                          nullptr, channels, qstep, quant, ctx->f_attr);
  if (rc != GSNFS_OK) return rc;
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_counts, ctx->f_counts, sizeof(gsnfs_counts), cudaMemcpyDeviceToHost, st));
  if (nv) {
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_voxel_xyz, ctx->f_vxyz, nv * 12, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_attr, ctx->f_attr, nv * C * 4, cudaMemcpyDeviceToHost, st));
  }
  GSNFS_CUDA_OK(ctx, cudaStreamSynchronize(st));
  return take_sticky(ctx);
}

// ---- the same two frame calls with the coefficients entropy coded (RLGR) before they leave the device ----------
static int frame_encode_host_packed_impl(gsnfs_ctx* ctx, gsnfs_stream stream, const float* h_xyz, const float* h_attr, uint64_t n,
                                   int channels, const float bbox_min[3], const float bbox_max[3], int depth,
                                   const float* qstep, const gsnfs_quant* quant, int rlgr_block, uint8_t* h_occ,
                                   uint64_t occ_capacity, uint32_t* h_level_sizes, uint32_t* h_weights,
                                   uint32_t* h_block_bits, uint8_t* h_stream, uint64_t stream_capacity,
                                   gsnfs_counts* h_counts, gsnfs_rlgr_info* h_info) {
  if (!ctx || !h_occ || !h_level_sizes || !h_counts || !h_info || !qstep ||
      (n && (!h_xyz || !h_attr || !h_weights || !h_block_bits || !h_stream)))
    return GSNFS_E_INVALID_ARGUMENT;
  if (n > ctx->max_points || channels > ctx->max_channels || channels < 1) return GSNFS_E_CAPACITY;
  if (rlgr_block < GSNFS_RLGR_MIN_BLOCK || rlgr_block > GSNFS_RLGR_MAX_BLOCK) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  int rc = frame_pool(ctx);
  if (rc != GSNFS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream, cs = ctx->copy_stream;
  const uint64_t cap = gsnfs_occ_capacity(n, depth);
  if (cap == 0 || occ_capacity < cap || cap > ctx->occ_cap) return depth < 1 || depth > GSNFS_MAX_DEPTH ? GSNFS_E_INVALID_ARGUMENT : GSNFS_E_CAPACITY;
  const size_t C = (size_t)channels;
  const uint64_t nbits = gsnfs_rlgr_blocks(n, channels, rlgr_block);
  // positions on the caller's stream, the (19x larger) attribute tensor on the copy stream: the position coder runs
  // while the attributes are still crossing PCIe
  GSNFS_CUDA_OK(ctx, cudaEventRecord(ctx->ev_a, st));                     // earlier work on st (previous frame) first
  GSNFS_CUDA_OK(ctx, cudaStreamWaitEvent(cs, ctx->ev_a, 0));
  if (n) {
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_xyz, h_xyz, n * 12, cudaMemcpyHostToDevice, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_attr, h_attr, n * C * 4, cudaMemcpyHostToDevice, cs));
  }
  GSNFS_CUDA_OK(ctx, cudaEventRecord(ctx->ev_b, cs));
  rc = gsnfs_octree_encode(ctx, stream, ctx->f_xyz, n, bbox_min, bbox_max, depth, ctx->f_occ, cap, ctx->f_levels,
                           ctx->f_perm, ctx->f_vkeys, ctx->f_vstart, ctx->f_counts);
  if (rc != GSNFS_OK) return rc;
  GSNFS_CUDA_OK(ctx, cudaStreamWaitEvent(st, ctx->ev_b, 0));
  rc = gsnfs_merge_raht_forward(ctx, stream, ctx->f_vkeys, ctx->f_perm, ctx->f_vstart, n, ctx->f_counts, depth, ctx->f_attr,
                                channels, qstep, quant, ctx->f_weights, ctx->f_q, nullptr);
  if (rc != GSNFS_OK) return rc;
  rc = gsnfs_rlgr_encode(ctx, stream, ctx->f_q, n, ctx->f_counts, channels, rlgr_block, ctx->f_bits, ctx->f_stream,
                         ctx->f_stream_cap < stream_capacity ? ctx->f_stream_cap : stream_capacity, ctx->f_info);
  if (rc != GSNFS_OK) return rc;
  // header first: the sizes of the remaining copies depend on it
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_counts, ctx->f_counts, sizeof(gsnfs_counts), cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_level_sizes, ctx->f_levels, sizeof(uint32_t) * (depth + 1), cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_info, ctx->f_info, sizeof(gsnfs_rlgr_info), cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaStreamSynchronize(st));
  const uint64_t nv = h_counts->n_voxels, ob = h_counts->occ_bytes;
  if (h_info->status) return GSNFS_E_CAPACITY;                            // stream buffer too small: nothing was written
  if (nv) {
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_occ, ctx->f_occ, ob, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_weights, ctx->f_weights, nv * 4, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_block_bits, ctx->f_bits, nbits * 4, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_stream, ctx->f_stream, h_info->stream_bytes, cudaMemcpyDeviceToHost, st));
    GSNFS_CUDA_OK(ctx, cudaStreamSynchronize(st));
  }
  return take_sticky(ctx);
}

static int frame_decode_host_packed_impl(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* h_occ, uint64_t occ_bytes,
                                   const uint32_t* level_sizes, int depth, const uint32_t* h_weights,
                                   const uint32_t* h_block_bits, const uint8_t* h_stream, uint64_t stream_bytes,
                                   int rlgr_block, int channels, const float* qstep, const gsnfs_quant* quant,
                                   uint32_t* h_voxel_xyz, float* h_attr, gsnfs_counts* h_counts) {
  if (!ctx || !level_sizes || !h_counts || !qstep) return GSNFS_E_INVALID_ARGUMENT;
  if (depth < 1 || depth > GSNFS_MAX_DEPTH) return GSNFS_E_INVALID_ARGUMENT;
  if (rlgr_block < GSNFS_RLGR_MIN_BLOCK || rlgr_block > GSNFS_RLGR_MAX_BLOCK) return GSNFS_E_INVALID_ARGUMENT;
  const uint64_t nv = level_sizes[depth];
  if (nv && (!h_occ || !h_block_bits || (!h_stream && stream_bytes) || !h_voxel_xyz || !h_attr)) return GSNFS_E_INVALID_ARGUMENT;
  if (nv > ctx->max_points || channels > ctx->max_channels || channels < 1 || occ_bytes + 1 > ctx->occ_cap)
    return GSNFS_E_CAPACITY;
  if (!octree_header_ok(level_sizes, depth, occ_bytes)) {
    h_counts->n_voxels = 0; h_counts->occ_bytes = (uint32_t)occ_bytes; h_counts->status = 1; h_counts->reserved = 0;
    return GSNFS_OK;
  }
  if (h_weights)
    for (uint64_t i = 0; i < nv; ++i)
      if (h_weights[i] == 0) return GSNFS_E_INVALID_ARGUMENT;
  GSNFS_ON_DEVICE(ctx);
  int rc = frame_pool(ctx);
  if (rc != GSNFS_OK) return rc;
  if (stream_bytes > ctx->f_stream_cap) return GSNFS_E_CAPACITY;
  cudaStream_t st = (cudaStream_t)stream, cs = ctx->copy_stream;
  const size_t C = (size_t)channels;
  const uint64_t nbits = gsnfs_rlgr_blocks(nv, channels, rlgr_block);
  GSNFS_CUDA_OK(ctx, cudaEventRecord(ctx->ev_a, st));
  GSNFS_CUDA_OK(ctx, cudaStreamWaitEvent(cs, ctx->ev_a, 0));
  if (nv) {
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_occ, h_occ, occ_bytes, cudaMemcpyHostToDevice, st));
    // the coefficient stream travels on the copy stream while the position decoder runs
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_bits, h_block_bits, nbits * 4, cudaMemcpyHostToDevice, cs));
    GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_stream, h_stream, stream_bytes, cudaMemcpyHostToDevice, cs));
    if (h_weights) GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(ctx->f_weights, h_weights, nv * 4, cudaMemcpyHostToDevice, cs));
  }
  GSNFS_CUDA_OK(ctx, cudaEventRecord(ctx->ev_b, cs));
  rc = gsnfs_octree_decode(ctx, stream, ctx->f_occ, occ_bytes, level_sizes, depth, ctx->f_vxyz, ctx->f_vkeys, ctx->f_counts);
  if (rc != GSNFS_OK) return rc;
  if (nv) GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_voxel_xyz, ctx->f_vxyz, nv * 12, cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaStreamWaitEvent(st, ctx->ev_b, 0));
  rc = gsnfs_rlgr_decode(ctx, stream, ctx->f_stream, stream_bytes, ctx->f_bits, nv, channels, rlgr_block, ctx->f_q, ctx->f_info);
  if (rc != GSNFS_OK) return rc;
  rc = gsnfs_raht_inverse(ctx, stream, ctx->f_vkeys, h_weights ? ctx->f_weights : nullptr, nv, ctx->f_counts, depth, ctx->f_q,
                          nullptr, channels, qstep, quant, ctx->f_attr);
  if (rc != GSNFS_OK) return rc;
  gsnfs_rlgr_info info;
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_counts, ctx->f_counts, sizeof(gsnfs_counts), cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(&info, ctx->f_info, sizeof(info), cudaMemcpyDeviceToHost, st));
  if (nv) GSNFS_CUDA_OK(ctx, cudaMemcpyAsync(h_attr, ctx->f_attr, nv * C * 4, cudaMemcpyDeviceToHost, st));
  GSNFS_CUDA_OK(ctx, cudaStreamSynchronize(st));
  if (info.status) h_counts->status |= 1u;                                 // a corrupt coefficient stream is a corrupt frame
  return take_sticky(ctx);
}

// A frame call that fails after its first cudaMemcpyAsync (a bad bbox found by gsnfs_octree_encode, a capacity error of
// a later stage, a CUDA error) must not hand the caller's pinned buffers back while a DMA still reads or writes them:
// every failing return drains both streams first.  Successful returns have synchronised already.
static int frame_done(gsnfs_ctx* ctx, gsnfs_stream stream, int rc) {
  if (rc != GSNFS_OK && ctx) {
    cudaStreamSynchronize((cudaStream_t)stream);
    if (ctx->fpool && ctx->copy_stream) cudaStreamSynchronize(ctx->copy_stream);
  }
  return rc;
}

int gsnfs_frame_encode_host(gsnfs_ctx* ctx, gsnfs_stream stream, const float* h_xyz, const float* h_attr, uint64_t n,
                            int channels, const float bbox_min[3], const float bbox_max[3], int depth,
                            const float* qstep, const gsnfs_quant* quant, uint8_t* h_occ, uint64_t occ_capacity,
                            uint32_t* h_level_sizes, uint32_t* h_weights, int32_t* h_qcoeff, gsnfs_counts* h_counts) {
  return frame_done(ctx, stream,
                    frame_encode_host_impl(ctx, stream, h_xyz, h_attr, n, channels, bbox_min, bbox_max, depth, qstep, quant, h_occ,
                                           occ_capacity, h_level_sizes, h_weights, h_qcoeff, h_counts));
}

int gsnfs_frame_decode_host(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* h_occ, uint64_t occ_bytes,
                            const uint32_t* level_sizes, int depth, const uint32_t* h_weights, const int32_t* h_qcoeff,
                            int channels, const float* qstep, const gsnfs_quant* quant, uint32_t* h_voxel_xyz,
                            float* h_attr, gsnfs_counts* h_counts) {
  return frame_done(ctx, stream,
                    frame_decode_host_impl(ctx, stream, h_occ, occ_bytes, level_sizes, depth, h_weights, h_qcoeff, channels, qstep, quant,
                                           h_voxel_xyz, h_attr, h_counts));
}

int gsnfs_frame_encode_host_packed(gsnfs_ctx* ctx, gsnfs_stream stream, const float* h_xyz, const float* h_attr, uint64_t n,
                                   int channels, const float bbox_min[3], const float bbox_max[3], int depth,
                                   const float* qstep, const gsnfs_quant* quant, int rlgr_block, uint8_t* h_occ,
                                   uint64_t occ_capacity, uint32_t* h_level_sizes, uint32_t* h_weights,
                                   uint32_t* h_block_bits, uint8_t* h_stream, uint64_t stream_capacity,
                                   gsnfs_counts* h_counts, gsnfs_rlgr_info* h_info) {
  return frame_done(ctx, stream,
                    frame_encode_host_packed_impl(ctx, stream, h_xyz, h_attr, n, channels, bbox_min, bbox_max, depth, qstep, quant, rlgr_block, h_occ,
                                                  occ_capacity, h_level_sizes, h_weights, h_block_bits, h_stream, stream_capacity, h_counts, h_info));
}

int gsnfs_frame_decode_host_packed(gsnfs_ctx* ctx, gsnfs_stream stream, const uint8_t* h_occ, uint64_t occ_bytes,
                                   const uint32_t* level_sizes, int depth, const uint32_t* h_weights,
                                   const uint32_t* h_block_bits, const uint8_t* h_stream, uint64_t stream_bytes,
                                   int rlgr_block, int channels, const float* qstep, const gsnfs_quant* quant,
                                   uint32_t* h_voxel_xyz, float* h_attr, gsnfs_counts* h_counts) {
  return frame_done(ctx, stream,
                    frame_decode_host_packed_impl(ctx, stream, h_occ, occ_bytes, level_sizes, depth, h_weights, h_block_bits, h_stream, stream_bytes,
                                                  rlgr_block, channels, qstep, quant, h_voxel_xyz, h_attr, h_counts));
}

}  // extern "C"
