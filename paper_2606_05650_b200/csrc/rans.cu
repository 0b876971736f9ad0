// Entropy coding of the octree occupancy bytes: static order-0 range-ANS (rANS), in place of the closed nvCOMP ANS the
// paper calls ("runs a GPU-based entropy encoder, ANS"; L283; L801 "adds only ~0.3 ms but roughly halves
// the compressed size").  Rules = reading [R17] of DESIGN.md: one 12-bit
// frequency table per frame, independent blocks of 1024 bytes, 32-bit state with lower bound 2^16 and 16-bit
// renormalisation words, a block = final state + words in decoder order.
//
// Five small launches: histogram -> model (one warp quantises the 256 counts to sum 4096) -> one thread per block
// encodes backwards from a padded shared-memory copy of its 1024 bytes into a strided scratch -> scan of the word counts
// -> compaction into the caller's payload.  Decoding is one launch: a 4096-entry slot -> symbol table in shared
// memory, one thread per block, output staged in shared memory and written coalesced.
#include <mutex>

#include "common.cuh"

namespace gsnfs {

namespace {

constexpr uint32_t kRansBlock = GSNFS_RANS_BLOCK;
constexpr uint32_t kRansM = 4096u;
constexpr uint32_t kRansL = 65536u;
constexpr int kRansCta = 32;                           // blocks (= threads) per CTA
constexpr uint32_t kRansPitch = kRansBlock + 4u;       // bytes per staged block: + 4 keeps the 32 threads on 32 banks
constexpr uint32_t kRansScratchWords = kRansBlock;     // a block never needs more than 12 bits per byte = 768 words

__global__ void __launch_bounds__(256) rans_hist_kernel(const uint8_t* __restrict__ data, uint64_t n_host,
                                                        const uint32_t* __restrict__ n_dev, uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_h[256];
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  s_h[threadIdx.x] = 0;
  __syncthreads();
  const uint64_t stride = (uint64_t)gridDim.x * 256u * 4u;
  for (uint64_t i = ((uint64_t)blockIdx.x * 256u + threadIdx.x) * 4u; i < n; i += stride) {
    if (i + 4 <= n) {
      const uint32_t w = *reinterpret_cast<const uint32_t*>(data + i);
      atomicAdd(&s_h[w & 0xffu], 1u); atomicAdd(&s_h[(w >> 8) & 0xffu], 1u);
      atomicAdd(&s_h[(w >> 16) & 0xffu], 1u); atomicAdd(&s_h[w >> 24], 1u);
    } else {
      for (uint64_t k = i; k < n; ++k) atomicAdd(&s_h[data[k]], 1u);
    }
  }
  __syncthreads();
  if (s_h[threadIdx.x]) atomicAdd(&hist[threadIdx.x], s_h[threadIdx.x]);
}

// one warp: lane l owns symbols 8l .. 8l+7
__global__ void __launch_bounds__(32) rans_model_kernel(const uint32_t* __restrict__ hist, uint64_t n_host,
                                                        const uint32_t* __restrict__ n_dev, uint16_t* __restrict__ freq) {
  const int lane = threadIdx.x;
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  uint32_t h[8], f[8];
  int sum = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    h[j] = hist[8 * lane + j];
    uint32_t v = 0;
    if (h[j]) { v = (uint32_t)((uint64_t)h[j] * kRansM / n); if (v == 0) v = 1; }
    f[j] = v;
    sum += (int)v;
  }
  sum = __reduce_add_sync(0xffffffffu, sum);
  int d = (int)kRansM - sum;
  if (n == 0) d = 0;
  if (d > 0) {      // to the most frequent symbol (largest count, lowest index)
    uint32_t best = 0; int bj = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) if (h[j] > best) { best = h[j]; bj = j; }
    const uint32_t gmax = __reduce_max_sync(0xffffffffu, best);
    const unsigned who = __ballot_sync(0xffffffffu, best == gmax);
    if (lane == __ffs(who) - 1) f[bj] += (uint32_t)d;
  }
  while (d < 0) {   // one at a time from the largest quantised frequency (lowest index among equals)
    uint32_t best = 0; int bj = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) if (f[j] > best) { best = f[j]; bj = j; }
    const uint32_t gmax = __reduce_max_sync(0xffffffffu, best);
    const unsigned who = __ballot_sync(0xffffffffu, best == gmax);
    if (lane == __ffs(who) - 1) f[bj] -= 1u;
    ++d;
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) freq[8 * lane + j] = (uint16_t)f[j];
}

__global__ void __launch_bounds__(kRansCta) rans_encode_kernel(const uint8_t* __restrict__ data, uint64_t n_host,
                                                               const uint32_t* __restrict__ n_dev,
                                                               const uint16_t* __restrict__ freq,
                                                               uint16_t* __restrict__ scratch /* nblk x kRansScratchWords */,
                                                               uint32_t* __restrict__ states, uint16_t* __restrict__ nwords,
                                                               uint64_t nblk_host) {
  extern __shared__ __align__(16) uint8_t s_data[];                 // kRansCta x kRansPitch
  __shared__ uint16_t s_f[256];
  __shared__ uint16_t s_cum[256];
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  const int t = threadIdx.x;
  for (int s = t; s < 256; s += kRansCta) s_f[s] = freq[s];
  __syncwarp();
  if (t == 0) { uint32_t c = 0; for (int s = 0; s < 256; ++s) { s_cum[s] = (uint16_t)c; c += s_f[s]; } }
  const uint64_t b0 = (uint64_t)blockIdx.x * kRansCta;
  const uint64_t base = b0 * kRansBlock;
  if (base >= n) { if (b0 + t < nblk_host) nwords[b0 + t] = 0; return; }
  const uint64_t span = min((uint64_t)kRansCta * kRansBlock, n - base);
  for (uint64_t i = (uint64_t)t * 4u; i < span; i += kRansCta * 4u) {      // coalesced, 4 bytes per lane
    const uint32_t blk = (uint32_t)(i / kRansBlock), o = (uint32_t)(i % kRansBlock);
    uint32_t w = 0;
    if (i + 4 <= span) w = *reinterpret_cast<const uint32_t*>(data + base + i);
    else for (uint64_t k = i; k < span; ++k) w |= (uint32_t)data[base + k] << (8 * (k - i));
    *reinterpret_cast<uint32_t*>(s_data + blk * kRansPitch + o) = w;
  }
  __syncwarp();
  const uint64_t myb = b0 + t;
  const uint64_t mybase = myb * kRansBlock;
  if (mybase >= n) { if (myb < nblk_host) nwords[myb] = 0; return; }
  const uint32_t cnt = (uint32_t)min((uint64_t)kRansBlock, n - mybase);
  const uint8_t* my = s_data + t * kRansPitch;
  uint16_t* out = scratch + myb * kRansScratchWords + kRansScratchWords;      // filled backwards: decoder order
  uint32_t nw = 0, x = kRansL;
  for (uint32_t i = cnt; i-- > 0;) {
    const uint32_t s = my[i], fs = s_f[s];
    if ((uint64_t)x >= ((uint64_t)fs << 20)) { *--out = (uint16_t)(x & 0xffffu); x >>= 16; ++nw; }
    const uint32_t q = x / fs;
    x = q * kRansM + (x - q * fs) + s_cum[s];
  }
  states[myb] = x;
  nwords[myb] = (uint16_t)nw;
}

// one CTA: offsets of the block streams (4 + 2 nwords bytes each); totals and overflow status
__global__ void __launch_bounds__(1024) rans_scan_kernel(const uint16_t* __restrict__ nwords, uint64_t n_host,
                                                         const uint32_t* __restrict__ n_dev, uint64_t nblk_host,
                                                         uint64_t* __restrict__ off, uint64_t capacity,
                                                         gsnfs_rlgr_info* __restrict__ info) {
  __shared__ uint64_t s_warp[33];
  const uint64_t n = n_dev ? min((uint64_t)*n_dev, n_host) : n_host;
  const uint64_t nblk = min(nblk_host, (n + kRansBlock - 1) / kRansBlock);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint64_t carry = 0;
  for (uint64_t base = 0; base < nblk_host; base += 1024) {
    const uint64_t i = base + tid;
    const uint64_t v = i < nblk ? 4ull + 2ull * nwords[i] : 0ull;
    uint64_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint64_t tt = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += tt;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      const uint64_t w = s_warp[lane];
      uint64_t winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint64_t tt = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += tt;
      }
      s_warp[lane] = winc - w;
      if (lane == 31) s_warp[32] = winc;
    }
    __syncthreads();
    if (i < nblk_host) off[i] = carry + s_warp[warp] + inc - v;
    carry += s_warp[32];
    __syncthreads();
  }
  if (tid == 0) {
    off[nblk_host] = carry;
    info->stream_bytes = carry;
    info->n_blocks = (uint32_t)nblk;
    info->status = carry > capacity ? 2u : 0u;
  }
}

__global__ void __launch_bounds__(128) rans_pack_kernel(const uint16_t* __restrict__ scratch, const uint32_t* __restrict__ states,
                                                        const uint16_t* __restrict__ nwords, const uint64_t* __restrict__ off,
                                                        uint8_t* __restrict__ payload, const gsnfs_rlgr_info* __restrict__ info) {
  const uint64_t b = blockIdx.x;
  if (info->status || b >= info->n_blocks) return;
  const uint32_t nw = nwords[b];
  uint8_t* dst = payload + off[b];
  if (threadIdx.x < 4) dst[threadIdx.x] = (uint8_t)(states[b] >> (8 * threadIdx.x));
  const uint16_t* src = scratch + b * kRansScratchWords + (kRansScratchWords - nw);
  for (uint32_t i = threadIdx.x; i < nw; i += 128) {
    const uint16_t w = src[i];
    dst[4 + 2 * i] = (uint8_t)w;
    dst[5 + 2 * i] = (uint8_t)(w >> 8);
  }
}

__global__ void __launch_bounds__(kRansCta) rans_decode_kernel(const uint8_t* __restrict__ payload, uint64_t payload_bytes,
                                                               const uint16_t* __restrict__ freq,
                                                               const uint16_t* __restrict__ nwords,
                                                               const uint64_t* __restrict__ off, uint64_t n,
                                                               uint8_t* __restrict__ out, gsnfs_rlgr_info* __restrict__ info) {
  extern __shared__ __align__(16) uint8_t s_dyn[];                  // kRansCta x kRansPitch output staging, then the slot table
  uint8_t* s_out = s_dyn;
  uint8_t* s_sym = s_dyn + kRansCta * kRansPitch;                   // kRansM
  __shared__ uint16_t s_f[256];
  __shared__ uint16_t s_cum[257];
  __shared__ uint32_t s_bad;
  const int t = threadIdx.x;
  for (int s = t; s < 256; s += kRansCta) s_f[s] = freq[s];
  if (t == 0) s_bad = 0;
  __syncwarp();
  if (t == 0) { uint32_t c = 0; for (int s = 0; s < 256; ++s) { s_cum[s] = (uint16_t)min(c, 65535u); c += s_f[s]; } s_cum[256] = (uint16_t)min(c, 65535u); if (c != kRansM) s_bad = 1; }
  __syncwarp();
  const bool model_ok = s_bad == 0;
  if (model_ok)
    for (int s = t; s < 256; s += kRansCta)
      for (uint32_t k = 0; k < s_f[s]; ++k) s_sym[s_cum[s] + k] = (uint8_t)s;
  __syncwarp();
  const uint64_t b0 = (uint64_t)blockIdx.x * kRansCta;
  const uint64_t base = b0 * kRansBlock;
  if (base >= n) return;
  const uint64_t myb = b0 + t, mybase = myb * kRansBlock;
  bool bad = !model_ok;
  if (mybase < n) {
    const uint32_t cnt = (uint32_t)min((uint64_t)kRansBlock, n - mybase);
    uint8_t* my = s_out + t * kRansPitch;
    const uint32_t nw = nwords[myb];
    const uint64_t o = off[myb];
    if (bad || o + 4ull + 2ull * nw > payload_bytes) {
      bad = true;
      for (uint32_t i = 0; i < cnt; ++i) my[i] = 0;
    } else {
      const uint8_t* p = payload + o;
      uint32_t x = (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24);
      uint32_t w = 0;
      for (uint32_t i = 0; i < cnt; ++i) {
        const uint32_t slot = x & (kRansM - 1u);
        const uint32_t s = s_sym[slot];
        my[i] = (uint8_t)s;
        x = (uint32_t)s_f[s] * (x >> 12) + slot - s_cum[s];
        if (x < kRansL) {
          uint32_t nxt = 0;
          if (w < nw) nxt = (uint32_t)p[4 + 2 * w] | ((uint32_t)p[5 + 2 * w] << 8); else bad = true;
          ++w;
          x = (x << 16) | nxt;
        }
      }
      if (w != nw || x != kRansL) bad = true;
    }
  }
  if (bad) atomicOr(&info->status, 1u);
  __syncwarp();
  const uint64_t span = min((uint64_t)kRansCta * kRansBlock, n - base);
  for (uint64_t i = t; i < span; i += kRansCta) out[base + i] = s_out[(i / kRansBlock) * kRansPitch + (i % kRansBlock)];
}

}  // namespace

int run_rans_encode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_data, uint64_t n, const uint32_t* n_dev, uint16_t* d_freq,
                    uint16_t* d_nwords, uint8_t* d_payload, uint64_t capacity, gsnfs_rlgr_info* d_info) {
  const uint64_t nblk = (n + kRansBlock - 1) / kRansBlock;
  if (nblk + kRansCta + 1 > ctx->rans_blocks_cap) return GSNFS_E_CAPACITY;
  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(ctx->rans_hist, 0, 256 * sizeof(uint32_t), st));
  const int hgrid = (int)min((uint64_t)ctx->num_sms * 4u, n / 1024 + 1);
  GSNFS_KERNEL(ctx, st, "rans_hist");
  rans_hist_kernel<<<hgrid, 256, 0, st>>>(d_data, n, n_dev, ctx->rans_hist);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "rans_model");
  rans_model_kernel<<<1, 32, 0, st>>>(ctx->rans_hist, n, n_dev, d_freq);
  GSNFS_LAUNCH_CHECK(ctx, st);
  const int egrid = (int)((nblk + kRansCta - 1) / kRansCta);
  if (egrid > 0) {
    GSNFS_KERNEL(ctx, st, "rans_encode");
    rans_encode_kernel<<<egrid, kRansCta, kRansCta * kRansPitch, st>>>(d_data, n, n_dev, d_freq, ctx->rans_scratch,
                                                                      ctx->rans_states, d_nwords, nblk);
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  GSNFS_KERNEL(ctx, st, "rans_scan");
  rans_scan_kernel<<<1, 1024, 0, st>>>(d_nwords, n, n_dev, nblk, ctx->rans_off, capacity, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  if (nblk) {
    GSNFS_KERNEL(ctx, st, "rans_pack");
    rans_pack_kernel<<<(unsigned)nblk, 128, 0, st>>>(ctx->rans_scratch, ctx->rans_states, d_nwords, ctx->rans_off, d_payload, d_info);
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  return GSNFS_OK;
}

int run_rans_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_payload, uint64_t payload_bytes, const uint16_t* d_freq,
                    const uint16_t* d_nwords, uint64_t n, uint8_t* d_out, gsnfs_rlgr_info* d_info) {
  const uint64_t nblk = (n + kRansBlock - 1) / kRansBlock;
  if (nblk + kRansCta + 1 > ctx->rans_blocks_cap) return GSNFS_E_CAPACITY;
  GSNFS_KERNEL(ctx, st, "rans_scan");
  rans_scan_kernel<<<1, 1024, 0, st>>>(d_nwords, n, nullptr, nblk, ctx->rans_off, ~0ull, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  const int grid = (int)((nblk + kRansCta - 1) / kRansCta);
  if (grid > 0) {
    GSNFS_KERNEL(ctx, st, "rans_decode");
    rans_decode_kernel<<<grid, kRansCta, kRansCta * kRansPitch + kRansM, st>>>(d_payload, payload_bytes, d_freq, d_nwords,
                                                                              ctx->rans_off, n, d_out, d_info);
    GSNFS_LAUNCH_CHECK(ctx, st);
  }
  return GSNFS_OK;
}

int rans_setup(gsnfs_ctx* ctx) {
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(rans_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(kRansCta * kRansPitch + kRansM)));
  GSNFS_CUDA_OK(ctx, cudaFuncSetAttribute(rans_encode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(kRansCta * kRansPitch)));
  return GSNFS_OK;
}

}  // namespace gsnfs

// ---- gsnfs_rans_decode_static: the decoder without a context and without any allocation ---------------------------
// For callers that must not allocate device memory (see gsnfs.h: the GPU belongs to the application's own pool, the
// memory budget is frozen, or a cudaMalloc's device-wide synchronisation has no place in their frame loop).  The one
// piece of working memory the decoder needs -- the byte offset of every block stream, which run_rans_decode() keeps in
// the context scratch -- lives here in a file-scope device array that ships inside the library image.  The kernels are
// the ones above; only where `off` points differs.

namespace gsnfs {
namespace {

constexpr uint64_t kStaticMaxBlocks = GSNFS_RANS_STATIC_MAX_BYTES / kRansBlock;      // 32768 blocks
static_assert(GSNFS_RANS_STATIC_MAX_BYTES % kRansBlock == 0, "limit is a whole number of blocks");

// 256 KB + 8 on every GPU that loads the library, until the process exits.  In HOST code this name is only a handle
// for cudaGetSymbolAddress(): it is not a device address and must never be handed to a kernel as one.
static __device__ __align__(256) uint64_t g_static_off[kStaticMaxBlocks + 1];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
uint64_t* g_static_off_dev[kStaticMaxDevices];     // device address of g_static_off on device i; nullptr = not set up

// Once per device, with that device current: resolve the array's device address (every device has its own copy of
// the array at its own address) and raise the decoder's dynamic shared memory limit as rans_setup() does per context.
int static_off_for_current_device(uint64_t** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices) return GSNFS_E_CUDA;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_off_dev[dev]) {
    uint64_t* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_static_off) != cudaSuccess || !p) return GSNFS_E_CUDA;
    if (cudaFuncSetAttribute(rans_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(kRansCta * kRansPitch + kRansM)) != cudaSuccess)
      return GSNFS_E_CUDA;
    g_static_off_dev[dev] = p;
  }
  *out = g_static_off_dev[dev];
  return GSNFS_OK;
}

}  // namespace
}  // namespace gsnfs

int gsnfs_rans_decode_static(gsnfs_stream stream, const uint8_t* d_payload, uint64_t payload_bytes,
                             const uint16_t* d_freq, const uint16_t* d_nwords, uint64_t n, uint8_t* d_out,
                             gsnfs_rans_info* d_info) {
  using namespace gsnfs;
  if (!d_freq || !d_info || (n && (!d_payload || !d_nwords || !d_out))) return GSNFS_E_INVALID_ARGUMENT;
  if (n >= (1ull << 32)) return GSNFS_E_INVALID_ARGUMENT;
  if (n > GSNFS_RANS_STATIC_MAX_BYTES) return GSNFS_E_CAPACITY;      // the built-in table has no room: nothing is enqueued
  uint64_t* off = nullptr;
  const int rc = static_off_for_current_device(&off);
  if (rc != GSNFS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const uint64_t nblk = (n + kRansBlock - 1) / kRansBlock;           // <= kStaticMaxBlocks; the scan writes off[0 .. nblk]
  // The scan rewrites every offset this call's decoder reads, and all of d_info, so the previous call's leftovers in
  // the table are never seen and nothing needs a memset.
  rans_scan_kernel<<<1, 1024, 0, st>>>(d_nwords, n, nullptr, nblk, off, ~0ull, d_info);
  if (cudaPeekAtLastError() != cudaSuccess) return GSNFS_E_CUDA;
  const int grid = (int)((nblk + kRansCta - 1) / kRansCta);
  if (grid > 0) {
    rans_decode_kernel<<<grid, kRansCta, kRansCta * kRansPitch + kRansM, st>>>(d_payload, payload_bytes, d_freq, d_nwords, off,
                                                                              n, d_out, d_info);
    if (cudaPeekAtLastError() != cudaSuccess) return GSNFS_E_CUDA;
  }
  return GSNFS_OK;
}
