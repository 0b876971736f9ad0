// Device-wide exclusive scan of uint32 values (reduce -> scan of tile sums -> down-sweep).
// Used for the leaf-weight prefix sums of the RAHT schedule ([R1]: W_l from prefix sums of the leaf
// weights, generalising Alg. A.4 l.8) and for the decoder's popcount -> exclusive prefix sum
// (Alg. A.2 l.7-10).  No inter-CTA waiting: three plain launches.
#include "common.cuh"

namespace gsnfs {

struct LoadU32 {
  const uint32_t* p;
  __device__ __forceinline__ void load8(uint32_t i0, uint32_t n, uint32_t v[8]) const {
    if (i0 + 8 <= n) {
      uint4 a = *reinterpret_cast<const uint4*>(p + i0);
      uint4 b = *reinterpret_cast<const uint4*>(p + i0 + 4);
      v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
      v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
    } else {
#pragma unroll
      for (int k = 0; k < 8; ++k) v[k] = (i0 + k < n) ? p[i0 + k] : 0u;
    }
  }
};

struct LoadPopc8 {
  const uint8_t* p;
  __device__ __forceinline__ void load8(uint32_t i0, uint32_t n, uint32_t v[8]) const {
    if (i0 + 8 <= n) {
      uint2 a = *reinterpret_cast<const uint2*>(p + i0);
#pragma unroll
      for (int k = 0; k < 4; ++k) v[k] = __popc((a.x >> (8 * k)) & 0xffu);
#pragma unroll
      for (int k = 0; k < 4; ++k) v[4 + k] = __popc((a.y >> (8 * k)) & 0xffu);
    } else {
#pragma unroll
      for (int k = 0; k < 8; ++k) v[k] = (i0 + k < n) ? __popc((unsigned)p[i0 + k]) : 0u;
    }
  }
};

template <typename Loader>
__global__ void __launch_bounds__(256) scan_reduce_kernel(Loader ld, uint32_t n_cap, const uint32_t* d_n,
                                                          uint32_t* __restrict__ sums) {
  __shared__ uint32_t s_w[8];
  const uint32_t n = d_n ? min(*d_n, n_cap) : n_cap;
  const uint32_t i0 = blockIdx.x * kScanTile + threadIdx.x * 8;
  uint32_t v[8];
  uint32_t s = 0;
  if (i0 < n) {
    ld.load8(i0, n, v);
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
  }
  s = __reduce_add_sync(0xffffffffu, s);
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) t += s_w[k];
    sums[blockIdx.x] = t;
  }
}

// In-place exclusive scan of the tile sums by one CTA of 1024 threads.
__global__ void __launch_bounds__(1024) scan_sums_kernel(uint32_t* __restrict__ sums, uint32_t ntiles) {
  __shared__ uint32_t s_w[33];
  __shared__ uint32_t s_carry;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (uint32_t base = 0; base < ntiles; base += 1024) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t v = i < ntiles ? sums[i] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      uint32_t w = s_w[lane], winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += t;
      }
      s_w[lane] = winc - w;
      if (lane == 31) s_w[32] = winc;
    }
    __syncthreads();
    const uint32_t carry = s_carry;
    if (i < ntiles) sums[i] = carry + s_w[warp] + inc - v;
    __syncthreads();
    if (threadIdx.x == 0) s_carry = carry + s_w[32];
    __syncthreads();
  }
}

template <typename Loader>
__global__ void __launch_bounds__(256) scan_down_kernel(Loader ld, uint32_t n_cap, const uint32_t* d_n,
                                                        const uint32_t* __restrict__ sums,
                                                        uint32_t* __restrict__ out) {
  __shared__ uint32_t s_w[9];
  const uint32_t n = d_n ? min(*d_n, n_cap) : n_cap;
  const uint32_t i0 = blockIdx.x * kScanTile + threadIdx.x * 8;
  if (blockIdx.x * (uint32_t)kScanTile > n) return;
  uint32_t v[8];
  uint32_t s = 0;
  if (i0 < n) {
    ld.load8(i0, n, v);
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
  } else {
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = 0;
  }
  uint32_t run = block_excl_scan_256(s, s_w, nullptr) + sums[blockIdx.x];
  if (i0 + 8 <= n) {
    uint4 a, b;
    a.x = run; run += v[0]; a.y = run; run += v[1]; a.z = run; run += v[2]; a.w = run; run += v[3];
    b.x = run; run += v[4]; b.y = run; run += v[5]; b.z = run; run += v[6]; b.w = run; run += v[7];
    *reinterpret_cast<uint4*>(out + i0) = a;
    *reinterpret_cast<uint4*>(out + i0 + 4) = b;
    if (i0 + 8 == n) out[n] = run;
  } else if (i0 <= n) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (i0 + k <= n) out[i0 + k] = run;
      run += v[k];
    }
  }
}

template <typename Loader>
static int run_scan(gsnfs_ctx* ctx, cudaStream_t st, Loader ld, uint32_t* d_out, uint32_t n_cap,
                    const uint32_t* d_n) {
  const uint32_t ntiles = n_cap / kScanTile + 1;
  if (ntiles > ctx->scan_tiles_cap) return GSNFS_E_CAPACITY;
  GSNFS_KERNEL(ctx, st, "scan_reduce");
  scan_reduce_kernel<Loader><<<ntiles, 256, 0, st>>>(ld, n_cap, d_n, ctx->scan_sums);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "scan_sums");
  scan_sums_kernel<<<1, 1024, 0, st>>>(ctx->scan_sums, ntiles);
  GSNFS_LAUNCH_CHECK(ctx, st);
  GSNFS_KERNEL(ctx, st, "scan_down");
  scan_down_kernel<Loader><<<ntiles, 256, 0, st>>>(ld, n_cap, d_n, ctx->scan_sums, d_out);
  GSNFS_LAUNCH_CHECK(ctx, st);
  return GSNFS_OK;
}

int run_scan_u32(gsnfs_ctx* ctx, cudaStream_t st, const uint32_t* d_in, uint32_t* d_out, uint32_t n_cap,
                 const uint32_t* d_n) {
  return run_scan(ctx, st, LoadU32{d_in}, d_out, n_cap, d_n);
}

int run_scan_popc8(gsnfs_ctx* ctx, cudaStream_t st, const uint8_t* d_in, uint32_t* d_out, uint32_t n) {
  return run_scan(ctx, st, LoadPopc8{d_in}, d_out, n, nullptr);
}

}  // namespace gsnfs
