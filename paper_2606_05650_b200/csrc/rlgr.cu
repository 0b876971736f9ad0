// Block-parallel adaptive Run-Length / Golomb-Rice coder for the quantised RAHT coefficients
// (section 3.4; L803 Appendix H "RLGR parallelization"; Table A.5): every attribute channel is
// cut into blocks of B consecutive coefficients, each block is an independent adaptive RLGR stream (fresh state), one
// GPU thread per block.  The coding rules are reading [R14] of DESIGN.md (the paper cites the coder only): sign
// folding u(x) = 2x / -2x-1; GR(u, kR) = unary quotient + kR remainder bits with a 32-ones escape; fixed-point adaptive
// parameters kP, kRP (L = 4, U0 = 3, D0 = 1, U1 = 2, D1 = 3), k = kP >> 2 selects "no run" (k = 0) or run mode with
// runs of 2^k zeros; start of a block kP = 0, kRP = 8; a 0 bit in run mode means min(2^k, coefficients left) zeros.
// Bits are MSB first; every block stream is padded to a multiple of 32 bits; block (b, c) is stored at position b*C + c.
//
// What differs from the paper's mapping (one thread per block of ONE channel over a channel-major copy): the threads of
// a CTA are the C channels of the SAME block of rows, so at every step they read C consecutive ints of the row-major
// (canonical) coefficient tensor -- coalesced, and no transposed copy of the tensor is ever made.  Encoding is
// count -> exclusive scan -> write: the first pass only measures every block, so streams are packed back to back with
// no worst-case slack and the caller's buffer is never overrun.
#include "common.cuh"

namespace gsnfs {

namespace {

constexpr int kRlgrBatch = 8;          // coefficients fetched ahead per thread (independent loads)

__device__ __forceinline__ uint32_t rlgr_fold(int32_t x) {
  return x >= 0 ? 2u * (uint32_t)x : 2u * (uint32_t)(-(int64_t)x) - 1u;
}
__device__ __forceinline__ int32_t rlgr_unfold(uint32_t u) {
  return (u & 1u) ? (int32_t)(-(int64_t)((u >> 1) + 1u)) : (int32_t)(u >> 1);
}
__device__ __forceinline__ uint32_t bswap32(uint32_t w) { return __byte_perm(w, 0u, 0x0123u); }

// MSB-first bit sink: WRITE = false only counts.
template <bool WRITE>
struct BitSink {
  uint64_t acc = 0;       // pending bits, left aligned
  uint32_t nb = 0;        // number of pending bits (< 32 between calls)
  uint64_t total = 0;
  uint32_t* out = nullptr;
  __device__ __forceinline__ void put(uint32_t v, uint32_t n) {      // n <= 32 low bits of v
    if (n == 0) return;
    total += n;
    if (WRITE) {
      acc |= (uint64_t)v << (64u - nb - n);
      nb += n;
      if (nb >= 32u) {
        *out++ = bswap32((uint32_t)(acc >> 32));
        acc <<= 32;
        nb -= 32u;
      }
    }
  }
  __device__ __forceinline__ void finish() {      // pad with zero bits to a multiple of 32
    const uint32_t pad = (uint32_t)((32u - (total & 31u)) & 31u);
    if (pad) put(0u, pad);
  }
};

template <bool WRITE>
__device__ __forceinline__ void gr_put(BitSink<WRITE>& s, uint32_t u, int& kRP) {
  const int kR = kRP >> 2;
  const uint32_t p = u >> kR;
  if (p < 32u) {
    s.put(((1u << p) - 1u) << 1, p + 1u);                       // p ones and a zero (p + 1 <= 32 bits)
    s.put(kR ? (u & ((1u << kR) - 1u)) : 0u, (uint32_t)kR);
    if (p == 0u) kRP = max(kRP - 2, 0);
    else if (p > 1u) kRP = min(kRP + (int)p + 1, 127);
  } else {
    s.put(0xffffffffu, 32u);
    s.put(u, 32u);
    kRP = min(kRP + 33, 127);
  }
}

// One CTA = the blocks (b, c) of one block of rows b, thread c = channel c.
// Offsets without a scan pass: the count pass leaves, per block row b, the bytes of its C streams (rowsum[b]) and, per
// 256 block rows, their sum (supersum).  Row b then starts at sum(supersum[0 .. b/256)) + sum(rowsum[256 (b/256) .. b)), and
// channel c inside the row at the exclusive prefix of the row's block sizes -- a few hundred cached loads per CTA.
constexpr uint32_t kRowGroup = 256;

struct RowOffsets { uint64_t row_start, total; };
// all threads of the CTA call it; nrows = block rows of the tensor (host upper bound)
__device__ RowOffsets rlgr_row_offsets(const uint64_t* __restrict__ rowsum, const uint64_t* __restrict__ supersum,
                                       uint32_t b, uint32_t nrows, uint64_t* s_red /* 2 */) {
  const uint32_t ng = (nrows + kRowGroup - 1) / kRowGroup, g = b / kRowGroup;
  uint64_t before = 0, total = 0;
  for (uint32_t i = threadIdx.x; i < ng; i += blockDim.x) { const uint64_t v = supersum[i]; total += v; if (i < g) before += v; }
  for (uint32_t i = g * kRowGroup + threadIdx.x; i < b; i += blockDim.x) before += rowsum[i];
  if (threadIdx.x == 0) { s_red[0] = 0; s_red[1] = 0; }
  __syncthreads();
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    before += __shfl_xor_sync(0xffffffffu, before, o);
    total += __shfl_xor_sync(0xffffffffu, total, o);
  }
  if ((threadIdx.x & 31) == 0) { atomicAdd((unsigned long long*)&s_red[0], before); atomicAdd((unsigned long long*)&s_red[1], total); }
  __syncthreads();
  RowOffsets r;
  r.row_start = s_red[0];
  r.total = s_red[1];
  return r;
}
// exclusive prefix over the threads of the CTA (blockDim.x <= 256) of one 32-bit value each; returns the CTA total too
__device__ __forceinline__ uint32_t cta_excl_scan(uint32_t v, uint32_t* s_w /* 9 */, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) s_w[warp] = inc;
  __syncthreads();
  uint32_t before = 0, tot = 0;
  for (int w = 0; w < nw; ++w) { const uint32_t x = s_w[w]; if (w < warp) before += x; tot += x; }
  *total = tot;
  return before + inc - v;
}

template <bool WRITE>
__global__ void __launch_bounds__(256) rlgr_encode_kernel(const int32_t* __restrict__ q, uint32_t n_host,
                                                          const uint32_t* __restrict__ n_dev, int C, uint32_t B,
                                                          uint32_t* __restrict__ block_bits, uint64_t* __restrict__ rowsum,
                                                          uint64_t* __restrict__ supersum, uint64_t capacity,
                                                          uint8_t* __restrict__ stream, gsnfs_rlgr_info* __restrict__ info) {
  __shared__ uint64_t s_red[2];
  __shared__ uint32_t s_w[9];
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const uint32_t b = blockIdx.x;
  const int c = threadIdx.x;
  const uint64_t r0 = (uint64_t)b * B;
  const bool active = c < C && r0 < n;
  if (!WRITE && r0 >= n) {               // block row beyond the actual N_v (n_host was an upper bound)
    if (c < C) block_bits[(size_t)b * C + c] = 0u;
    if (c == 0) rowsum[b] = 0ull;
    return;
  }
  uint64_t my_off = 0;
  if (WRITE) {
    if (r0 >= n) {                       // block 0 gets here only if the device-side N_v is 0: an empty stream, reported as such
      if (b == 0 && c == 0) { info->stream_bytes = 0ull; info->n_blocks = gridDim.x * (uint32_t)C; info->status = 0u; }
      return;
    }
    const RowOffsets ro = rlgr_row_offsets(rowsum, supersum, b, gridDim.x, s_red);
    uint32_t rtot;
    const uint32_t ex = cta_excl_scan(c < C ? block_bits[(size_t)b * C + c] >> 3 : 0u, s_w, &rtot);
    my_off = ro.row_start + ex;
    if (b == 0 && c == 0) {
      info->stream_bytes = ro.total;
      info->n_blocks = gridDim.x * (uint32_t)C;
      info->status = ro.total > capacity ? 2u : 0u;
    }
    if (ro.total > capacity) return;     // the stream does not fit the caller's buffer: nothing is written
  }
  if (!active && WRITE) return;
  const uint32_t cnt = active ? (uint32_t)min((uint64_t)B, (uint64_t)n - r0) : 0u;
  BitSink<WRITE> s;
  if (WRITE) s.out = reinterpret_cast<uint32_t*>(stream + my_off);
  const int32_t* src = q + r0 * C + c;
  int kP = 0, kRP = 8;
  uint32_t run = 0;
  for (uint32_t i0 = 0; i0 < cnt; i0 += kRlgrBatch) {
    int32_t v[kRlgrBatch];
#pragma unroll
    for (int j = 0; j < kRlgrBatch; ++j) v[j] = (i0 + j < cnt) ? __ldg(src + (size_t)(i0 + j) * C) : 0;
#pragma unroll
    for (int j = 0; j < kRlgrBatch; ++j) {
      if (i0 + j >= cnt) break;
      const int32_t x = v[j];
      const int k = kP >> 2;
      if (k == 0) {
        gr_put(s, rlgr_fold(x), kRP);
        kP = x == 0 ? min(kP + 3, 64) : max(kP - 1, 0);
      } else if (x == 0) {
        if (++run == (1u << k)) { s.put(0u, 1u); run = 0; kP = min(kP + 2, 64); }
      } else {
        s.put(1u, 1u);
        s.put(run, (uint32_t)k);
        run = 0;
        gr_put(s, rlgr_fold(x) - 1u, kRP);
        kP = max(kP - 3, 0);
      }
    }
  }
  if (run > 0) s.put(0u, 1u);
  s.finish();
  if (!WRITE) {
    if (active) block_bits[(size_t)b * C + c] = (uint32_t)s.total;
    uint32_t rtot;
    (void)cta_excl_scan(active ? (uint32_t)(s.total >> 3) : 0u, s_w, &rtot);
    if (c == 0) {
      rowsum[b] = rtot;
      atomicAdd((unsigned long long*)&supersum[b / kRowGroup], (unsigned long long)rtot);
    }
  }
}

// decoder side: the same two sums from the stream header
__global__ void __launch_bounds__(256) rlgr_rowsum_kernel(const uint32_t* __restrict__ block_bits, int C,
                                                          uint64_t* __restrict__ rowsum, uint64_t* __restrict__ supersum) {
  __shared__ uint32_t s_w[9];
  const uint32_t b = blockIdx.x;
  const int c = threadIdx.x;
  uint32_t rtot;
  (void)cta_excl_scan(c < C ? block_bits[(size_t)b * C + c] >> 3 : 0u, s_w, &rtot);
  if (c == 0) {
    rowsum[b] = rtot;
    atomicAdd((unsigned long long*)&supersum[b / kRowGroup], (unsigned long long)rtot);
  }
}

// MSB-first bit source over big-endian 32-bit words with a hard end: reading past it sets `bad`.
struct BitSource {
  const uint32_t* p;
  const uint32_t* end;
  uint64_t buf = 0;       // left aligned
  uint32_t avail = 0;
  uint32_t used = 0;      // bits consumed so far
  uint32_t limit = 0;     // bits in the block stream
  bool bad = false;
  __device__ __forceinline__ void refill() {
    if (avail <= 32u) {
      uint32_t w = 0u;
      if (p < end) w = bswap32(__ldg(p));
      ++p;
      buf |= (uint64_t)w << (32u - avail);
      avail += 32u;
    }
  }
  __device__ __forceinline__ uint32_t get(uint32_t n) {      // n <= 32
    if (n == 0) return 0u;
    refill();
    const uint32_t v = (uint32_t)(buf >> (64u - n));
    buf <<= n;
    avail -= n;
    used += n;
    return v;
  }
  __device__ __forceinline__ void check() { if (used > limit) bad = true; }     // a bit beyond the block's stream was consumed
};

__device__ __forceinline__ uint32_t gr_get(BitSource& s, int& kRP) {
  const int kR = kRP >> 2;
  s.refill();
  const uint32_t p = (uint32_t)__clz((int)~(uint32_t)(s.buf >> 32));       // leading ones of the next 32 bits
  uint32_t u;
  if (p < 32u) {
    s.buf <<= (p + 1u);
    s.avail -= (p + 1u);
    s.used += p + 1u;
    u = (p << kR) | s.get((uint32_t)kR);
    if (p == 0u) kRP = max(kRP - 2, 0);
    else if (p > 1u) kRP = min(kRP + (int)p + 1, 127);
  } else {
    s.buf <<= 32;
    s.avail -= 32u;
    s.used += 32u;
    u = s.get(32u);
    kRP = min(kRP + 33, 127);
  }
  return u;
}

__global__ void __launch_bounds__(256) rlgr_decode_kernel(const uint8_t* __restrict__ stream, uint64_t stream_bytes,
                                                          const uint32_t* __restrict__ block_bits,
                                                          const uint64_t* __restrict__ rowsum,
                                                          const uint64_t* __restrict__ supersum, uint32_t n, int C, uint32_t B,
                                                          int32_t* __restrict__ q, gsnfs_rlgr_info* __restrict__ info) {
  __shared__ uint64_t s_red[2];
  __shared__ uint32_t s_w[9];
  const uint32_t b = blockIdx.x;
  const int c = threadIdx.x;
  const uint64_t r0 = (uint64_t)b * B;
  const RowOffsets ro = rlgr_row_offsets(rowsum, supersum, b, gridDim.x, s_red);
  uint32_t rtot;
  const uint32_t ex = cta_excl_scan(c < C ? block_bits[(size_t)b * C + c] >> 3 : 0u, s_w, &rtot);
  if (b == 0 && c == 0) { info->stream_bytes = ro.total; info->n_blocks = gridDim.x * (uint32_t)C; }
  if (c >= C || r0 >= n) return;
  const uint32_t cnt = (uint32_t)min((uint64_t)B, (uint64_t)n - r0);
  const size_t e = (size_t)b * C + c;
  const uint64_t off = ro.row_start + ex, bytes = block_bits[e] >> 3;
  int32_t* dst = q + r0 * C + c;
  // header inconsistent with the stream: a length that is not whole words, a block that therefore starts off a word
  // boundary (some EARLIER entry was damaged: the word loads below would fault), or bytes beyond the stream
  if ((block_bits[e] & 31u) || (off & 3ull) || off + bytes > stream_bytes) {
    atomicOr(&info->status, 1u);
    for (uint32_t i = 0; i < cnt; ++i) dst[(size_t)i * C] = 0;
    return;
  }
  BitSource s;
  s.p = reinterpret_cast<const uint32_t*>(stream + off);
  s.end = s.p + (bytes >> 2);
  s.limit = block_bits[e];
  int kP = 0, kRP = 8;
  uint32_t i = 0;
  while (i < cnt) {
    const int k = kP >> 2;
    if (k == 0) {
      const int32_t x = rlgr_unfold(gr_get(s, kRP));
      dst[(size_t)i++ * C] = x;
      kP = x == 0 ? min(kP + 3, 64) : max(kP - 1, 0);
    } else if (s.get(1u) == 0u) {
      const uint32_t m = min(1u << k, cnt - i);
      for (uint32_t j = 0; j < m; ++j) dst[(size_t)i++ * C] = 0;
      kP = min(kP + 2, 64);
    } else {
      const uint32_t run = s.get((uint32_t)k);
      const uint32_t m = min(run, cnt - i);
      for (uint32_t j = 0; j < m; ++j) dst[(size_t)i++ * C] = 0;
      if (i >= cnt) { s.bad = true; break; }
      dst[(size_t)i++ * C] = rlgr_unfold(gr_get(s, kRP) + 1u);
      kP = max(kP - 3, 0);
    }
    s.check();
    if (s.bad) break;
  }
  for (; i < cnt; ++i) dst[(size_t)i * C] = 0;
  if (s.bad) atomicOr(&info->status, 1u);
}

__global__ void rlgr_info_kernel(gsnfs_rlgr_info* info, uint64_t bytes, uint32_t nblocks, uint32_t status) {
  info->stream_bytes = bytes;
  info->n_blocks = nblocks;
  info->status = status;
}

}  // namespace

int run_rlgr_encode(gsnfs_ctx* ctx, cudaStream_t st, const int32_t* d_q, uint32_t n, const gsnfs_counts* d_counts,
                    int channels, uint32_t block, uint32_t* d_block_bits, uint8_t* d_stream, uint64_t capacity,
                    gsnfs_rlgr_info* d_info) {
  const uint32_t nblk = (n + block - 1) / block;
  if (nblk + 1 > ctx->rlgr_rows_cap) return GSNFS_E_CAPACITY;
  if (n == 0) {
    GSNFS_KERNEL(ctx, st, "rlgr_info");
    rlgr_info_kernel<<<1, 1, 0, st>>>(d_info, 0ull, 0u, 0u);
    GSNFS_LAUNCH_CHECK(ctx, st);
    return GSNFS_OK;
  }
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const int threads = (channels + 31) & ~31;
  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(ctx->rlgr_supersum, 0, sizeof(uint64_t) * (nblk / kRowGroup + 1), st));
  GSNFS_KERNEL(ctx, st, "rlgr_count");
  rlgr_encode_kernel<false><<<nblk, threads, 0, st>>>(d_q, n, n_dev, channels, block, d_block_bits, ctx->rlgr_rowsum,
                                                      ctx->rlgr_supersum, 0ull, nullptr, nullptr);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "rlgr_write");
  rlgr_encode_kernel<true><<<nblk, threads, 0, st>>>(d_q, n, n_dev, channels, block, d_block_bits, ctx->rlgr_rowsum,
                                                     ctx->rlgr_supersum, capacity, d_stream, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

int run_rlgr_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_stream, uint64_t stream_bytes,
                    const uint32_t* d_block_bits, uint32_t n, int channels, uint32_t block, int32_t* d_q,
                    gsnfs_rlgr_info* d_info) {
  const uint32_t nblk = (n + block - 1) / block;
  if (nblk + 1 > ctx->rlgr_rows_cap) return GSNFS_E_CAPACITY;
  GSNFS_KERNEL(ctx, st, "rlgr_info");
  rlgr_info_kernel<<<1, 1, 0, st>>>(d_info, 0ull, 0u, (n == 0 && stream_bytes) ? 1u : 0u);
  GSNFS_LAUNCH_CHECK(ctx, st);
  if (n == 0) return GSNFS_OK;
  const int threads = (channels + 31) & ~31;
  GSNFS_CUDA_OK(ctx, cudaMemsetAsync(ctx->rlgr_supersum, 0, sizeof(uint64_t) * (nblk / kRowGroup + 1), st));
  GSNFS_KERNEL(ctx, st, "rlgr_rowsum");
  rlgr_rowsum_kernel<<<nblk, threads, 0, st>>>(d_block_bits, channels, ctx->rlgr_rowsum, ctx->rlgr_supersum);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "rlgr_decode");
  rlgr_decode_kernel<<<nblk, threads, 0, st>>>(d_stream, stream_bytes, d_block_bits, ctx->rlgr_rowsum, ctx->rlgr_supersum, n,
                                               channels, block, d_q, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

}  // namespace gsnfs
