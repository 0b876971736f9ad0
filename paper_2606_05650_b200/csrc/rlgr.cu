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
template <bool WRITE>
__global__ void __launch_bounds__(256) rlgr_encode_kernel(const int32_t* __restrict__ q, uint32_t n_host,
                                                          const uint32_t* __restrict__ n_dev, int C, uint32_t B,
                                                          uint32_t* __restrict__ block_bits,
                                                          const uint64_t* __restrict__ block_off,
                                                          uint8_t* __restrict__ stream, const gsnfs_rlgr_info* __restrict__ info) {
  const uint32_t n = n_dev ? min(*n_dev, n_host) : n_host;
  const uint32_t b = blockIdx.x;
  const int c = threadIdx.x;
  const uint64_t r0 = (uint64_t)b * B;
  if (c >= C) return;
  if (r0 >= n) {                         // block row beyond the actual N_v (n_host was an upper bound)
    if (!WRITE) block_bits[(size_t)b * C + c] = 0u;
    return;
  }
  if (WRITE && info->status) return;     // the stream does not fit the caller's buffer: nothing is written
  const uint32_t cnt = (uint32_t)min((uint64_t)B, (uint64_t)n - r0);
  BitSink<WRITE> s;
  if (WRITE) s.out = reinterpret_cast<uint32_t*>(stream + block_off[(size_t)b * C + c]);
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
  if (!WRITE) block_bits[(size_t)b * C + c] = (uint32_t)s.total;
}

// one CTA: exclusive scan of the block sizes (bytes) -> offsets; total, block count, overflow status
__global__ void __launch_bounds__(1024) rlgr_scan_kernel(const uint32_t* __restrict__ block_bits, uint64_t nent,
                                                         uint64_t* __restrict__ block_off, uint64_t capacity,
                                                         gsnfs_rlgr_info* __restrict__ info) {
  __shared__ uint64_t s_warp[33];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint64_t carry = 0;
  for (uint64_t base = 0; base < nent; base += 1024) {
    const uint64_t i = base + tid;
    const uint64_t v = i < nent ? (uint64_t)(block_bits[i] >> 3) : 0ull;
    uint64_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      const uint64_t w = s_warp[lane];
      uint64_t winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint64_t t = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += t;
      }
      s_warp[lane] = winc - w;
      if (lane == 31) s_warp[32] = winc;
    }
    __syncthreads();
    if (i < nent) block_off[i] = carry + s_warp[warp] + inc - v;
    carry += s_warp[32];
    __syncthreads();
  }
  if (tid == 0) {
    block_off[nent] = carry;
    info->stream_bytes = carry;
    info->n_blocks = (uint32_t)nent;
    info->status = carry > capacity ? 2u : 0u;
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
                                                          const uint64_t* __restrict__ block_off, uint32_t n, int C, uint32_t B,
                                                          int32_t* __restrict__ q, gsnfs_rlgr_info* __restrict__ info) {
  const uint32_t b = blockIdx.x;
  const int c = threadIdx.x;
  const uint64_t r0 = (uint64_t)b * B;
  if (c >= C || r0 >= n) return;
  const uint32_t cnt = (uint32_t)min((uint64_t)B, (uint64_t)n - r0);
  const size_t e = (size_t)b * C + c;
  const uint64_t off = block_off[e], bytes = block_bits[e] >> 3;
  int32_t* dst = q + r0 * C + c;
  if ((block_bits[e] & 31u) || off + bytes > stream_bytes) {      // header inconsistent with the stream
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
  const uint64_t nent = (uint64_t)nblk * (uint64_t)channels;
  if (nent + 1 > ctx->rlgr_off_cap) return GSNFS_E_CAPACITY;
  if (n == 0) {
    GSNFS_KERNEL(ctx, st, "rlgr_info");
    rlgr_info_kernel<<<1, 1, 0, st>>>(d_info, 0ull, 0u, 0u);
    GSNFS_LAUNCH_CHECK(ctx, st);
    return GSNFS_OK;
  }
  const uint32_t* n_dev = d_counts ? &d_counts->n_voxels : nullptr;
  const int threads = (channels + 31) & ~31;
  GSNFS_KERNEL(ctx, st, "rlgr_count");
  rlgr_encode_kernel<false><<<nblk, threads, 0, st>>>(d_q, n, n_dev, channels, block, d_block_bits, nullptr, nullptr, nullptr);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "rlgr_scan");
  rlgr_scan_kernel<<<1, 1024, 0, st>>>(d_block_bits, nent, ctx->rlgr_off, capacity, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "rlgr_write");
  rlgr_encode_kernel<true><<<nblk, threads, 0, st>>>(d_q, n, n_dev, channels, block, d_block_bits, ctx->rlgr_off, d_stream, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

int run_rlgr_decode(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_stream, uint64_t stream_bytes,
                    const uint32_t* d_block_bits, uint32_t n, int channels, uint32_t block, int32_t* d_q,
                    gsnfs_rlgr_info* d_info) {
  const uint32_t nblk = (n + block - 1) / block;
  const uint64_t nent = (uint64_t)nblk * (uint64_t)channels;
  if (nent + 1 > ctx->rlgr_off_cap) return GSNFS_E_CAPACITY;
  if (n == 0) {
    GSNFS_KERNEL(ctx, st, "rlgr_info");
    rlgr_info_kernel<<<1, 1, 0, st>>>(d_info, 0ull, 0u, stream_bytes ? 1u : 0u);
    GSNFS_LAUNCH_CHECK(ctx, st);
    return GSNFS_OK;
  }
  GSNFS_KERNEL(ctx, st, "rlgr_scan");
  rlgr_scan_kernel<<<1, 1024, 0, st>>>(d_block_bits, nent, ctx->rlgr_off, ~0ull, d_info);      // offsets from the header
  GSNFS_LAUNCH_CHECK(ctx, st);
  const int threads = (channels + 31) & ~31;
  GSNFS_KERNEL(ctx, st, "rlgr_decode");
  rlgr_decode_kernel<<<nblk, threads, 0, st>>>(d_stream, stream_bytes, d_block_bits, ctx->rlgr_off, n, channels, block, d_q, d_info);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

}  // namespace gsnfs
