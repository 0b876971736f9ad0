// Arithmetic shared by the RAHT transform kernels (raht.cu: generic kernels; raht_pipe.cu: the TMA-pipelined kernels):
// PTX helpers, packed fp32x2 butterflies, the dead-zone quantiser [R10] and its inverse.
#pragma once
#include "raht.cuh"

namespace gsnfs {

struct QStepParams {
  float step[GSNFS_MAX_CHANNELS];
};

// ---- small PTX helpers -----------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gmem_src) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(s), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// pull one C-float row (not necessarily line aligned) into L2
__device__ __forceinline__ void prefetch_row_l2(const float* row, int C) {
  const char* b = reinterpret_cast<const char*>(row);
  const char* e = b + (size_t)C * 4 - 1;
  for (const char* q = (const char*)((uintptr_t)b & ~(uintptr_t)127); q <= e; q += 128) prefetch_l2(q);
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// ---- TMA 1-D bulk store of a finished tile (rows are 16-byte multiples when C % 4 == 0) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int VEC> struct RowVec;
template <> struct RowVec<4> { using type = float4; };
template <> struct RowVec<1> { using type = float; };

// packed fp32x2 arithmetic (FFMA2 / FMUL2 / FADD2 on sm_100: one issue slot for two lanes of a float4); every
// product is rounded once and the sum is an FMA, exactly as the scalar fmaf(a, y0, b * y1) form
__device__ __forceinline__ uint64_t pk2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void upk2(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ float4 bf_lo(float a, float b, float4 y0, float4 y1) {      // a y0 + b y1
  const uint64_t aa = pk2(a, a), bb = pk2(b, b);
  float4 r;
  upk2(fma2(aa, pk2(y0.x, y0.y), mul2(bb, pk2(y1.x, y1.y))), r.x, r.y);
  upk2(fma2(aa, pk2(y0.z, y0.w), mul2(bb, pk2(y1.z, y1.w))), r.z, r.w);
  return r;
}
__device__ __forceinline__ float4 bf_hi(float a, float b, float4 y0, float4 y1) {      // a y1 - b y0
  const uint64_t aa = pk2(a, a), nb = pk2(-b, -b);
  float4 r;
  upk2(fma2(aa, pk2(y1.x, y1.y), mul2(nb, pk2(y0.x, y0.y))), r.x, r.y);
  upk2(fma2(aa, pk2(y1.z, y1.w), mul2(nb, pk2(y0.z, y0.w))), r.z, r.w);
  return r;
}
__device__ __forceinline__ float bf_lo(float a, float b, float y0, float y1) { return fmaf(a, y0, b * y1); }
__device__ __forceinline__ float bf_hi(float a, float b, float y0, float y1) { return fmaf(a, y1, -b * y0); }
__device__ __forceinline__ float4 vscale(float4 v, double s) {
  return make_float4((float)((double)v.x * s), (float)((double)v.y * s), (float)((double)v.z * s), (float)((double)v.w * s));
}
__device__ __forceinline__ float vscale(float v, double s) { return (float)((double)v * s); }

// Dead-zone quantiser [R10].  Definition (both sides of the parity test): q = sign(y) floor(|y| * (1/step) + f),
// evaluated in fp64 on the fp32 coefficient, saturating to int32 (quant_exact).  quant_fast2 evaluates the
// signed, half-shifted value t' = y * inv32 + sign(y)(f - 1/2) in fp32 and rounds it to nearest with the
// 1.5*2^23 magic constant, so that RN(t') = sign(y) floor(|y| inv + f) whenever t' is not within `guard` of a
// half-integer.  |t'_32 - t'_exact| <= 1.2e-7 |t| + 2e-8 (inv32 rounding, (f - 1/2) rounding, the FMA rounding);
// the guard 4e-7 |t'| + 4e-7 covers it with margin and |t'| >= 2^20 fails the test by itself.  Outside the guard
// the caller falls back to quant_exact, so the result always equals the fp64 definition.  Two values per call:
// the arithmetic is packed fp32x2.
__device__ __forceinline__ int quant_exact(float y, double inv, double f) {
  double m = floor(__dadd_rn(__dmul_rn(fabs((double)y), inv), f));      // product and sum rounded once each, no FMA (gsnfs.h)
  m = fmin(m, 2147483647.0);
  const int q = (int)m;
  return y < 0.f ? -q : (y > 0.f ? q : 0);      // sign(+-0) = 0: with dz_round == 1 the floor is 1 for y == 0, q is not
}
__device__ __forceinline__ bool quant_fast2(float y0, float y1, float i0, float i1, float fm, int& q0, int& q1) {
  const float s0 = __uint_as_float(__float_as_uint(fm) ^ (__float_as_uint(y0) & 0x80000000u));
  const float s1 = __uint_as_float(__float_as_uint(fm) ^ (__float_as_uint(y1) & 0x80000000u));
  const uint64_t t = fma2(pk2(y0, y1), pk2(i0, i1), pk2(s0, s1));
  const uint64_t u = add2(t, pk2(12582912.0f, 12582912.0f));
  const uint64_t rn = add2(u, pk2(-12582912.0f, -12582912.0f));
  const uint64_t d = fma2(t, pk2(-1.0f, -1.0f), rn);      // rn - t (exact); only |d| is used
  float t0, t1, u0, u1, d0, d1;
  upk2(t, t0, t1); upk2(u, u0, u1); upk2(d, d0, d1);
  q0 = __float_as_int(u0) - 0x4B400000;
  q1 = __float_as_int(u1) - 0x4B400000;
  const float lim0 = fmaf(fabsf(t0), -4e-7f, 0.4999996f), lim1 = fmaf(fabsf(t1), -4e-7f, 0.4999996f);
  return (fabsf(d0) < lim0) && (fabsf(d1) < lim1);
}
__device__ __forceinline__ float dequant1(int q, double step, double bias) {
  if (q == 0) return 0.f;
  const double m = fabs((double)q) + bias;
  return (float)(q < 0 ? -m * step : m * step);
}
// bias == 0 and |q| < 2^24: (float)q * step32 is the single rounding of the exact product = the fp64 result
__device__ __forceinline__ float dequant_fast(int q, float step32) { return (float)q * step32; }

struct QuantTab {          // per-channel constants in shared memory
  double* inv64;           // 1 / step            (forward)   |  step   (inverse)
  float* inv32;            // (float)(1 / step)   (forward)   |  step32 (inverse)
};

__device__ __forceinline__ int4 quant4(float4 y, int c4, const QuantTab& qt, double dz, float fm) {
  int4 q;
  const float4 iv = reinterpret_cast<const float4*>(qt.inv32)[c4];
  bool ok = quant_fast2(y.x, y.y, iv.x, iv.y, fm, q.x, q.y);
  ok &= quant_fast2(y.z, y.w, iv.z, iv.w, fm, q.z, q.w);
  if (!ok) {
    q.x = quant_exact(y.x, qt.inv64[4 * c4 + 0], dz); q.y = quant_exact(y.y, qt.inv64[4 * c4 + 1], dz);
    q.z = quant_exact(y.z, qt.inv64[4 * c4 + 2], dz); q.w = quant_exact(y.w, qt.inv64[4 * c4 + 3], dz);
  }
  return q;
}
__device__ __forceinline__ int quant1s(float y, int c, const QuantTab& qt, double dz, float fm) {
  int q0, q1;
  if (!quant_fast2(y, 0.f, qt.inv32[c], 0.f, fm, q0, q1)) q0 = quant_exact(y, qt.inv64[c], dz);
  return q0;
}

template <int VEC>
__device__ __forceinline__ void store_coeff(const float* row_s, int c, int C, size_t orow, const QuantTab& qt, double dz,
                                            float dz32, int32_t* out_q, float* out_f) {
  if constexpr (VEC == 4) {
    const float4 y = reinterpret_cast<const float4*>(row_s)[c];
    if (out_f) reinterpret_cast<float4*>(out_f + orow * C)[c] = y;
    if (out_q) reinterpret_cast<int4*>(out_q + orow * C)[c] = quant4(y, c, qt, dz, dz32);
  } else {
    const float y = row_s[c];
    if (out_f) out_f[orow * C + c] = y;
    if (out_q) out_q[orow * C + c] = quant1s(y, c, qt, dz, dz32);
  }
}

// i / d for i < 2^16 and d >= 1: umulhi(i, ceil(2^32 / d)), with d == 1 handled apart (the magic would be 2^32)
__device__ __forceinline__ uint32_t make_div_magic(uint32_t d) { return d > 1 ? (uint32_t)((0x100000000ull + d - 1) / d) : 0u; }
__device__ __forceinline__ uint32_t div_cv(uint32_t i, uint32_t magic, uint32_t d) { return d > 1 ? __umulhi(i, magic) : i; }

template <int VEC>
__device__ __forceinline__ void dequant_row_inplace(float* row_s, int c, const QuantTab& qt, double bias) {
  if constexpr (VEC == 4) {
    const int4 q = reinterpret_cast<const int4*>(row_s)[c];
    const int amax = max(max(abs(q.x), abs(q.y)), max(abs(q.z), abs(q.w)));
    const bool fast = bias == 0.0 && amax < (1 << 24);
    float4 y;
    if (fast) {
      const float4 st = reinterpret_cast<const float4*>(qt.inv32)[c];
      y = make_float4(dequant_fast(q.x, st.x), dequant_fast(q.y, st.y), dequant_fast(q.z, st.z), dequant_fast(q.w, st.w));
    } else {
      y = make_float4(dequant1(q.x, qt.inv64[4 * c + 0], bias), dequant1(q.y, qt.inv64[4 * c + 1], bias),
                      dequant1(q.z, qt.inv64[4 * c + 2], bias), dequant1(q.w, qt.inv64[4 * c + 3], bias));
    }
    reinterpret_cast<float4*>(row_s)[c] = y;
  } else {
    const int q = reinterpret_cast<const int*>(row_s)[c];
    row_s[c] = (bias == 0.0 && abs(q) < (1 << 24)) ? dequant_fast(q, qt.inv32[c]) : dequant1(q, qt.inv64[c], bias);
  }
}

}  // namespace gsnfs
