// r360 -- positional encoding of the bf16 tensor path (step a6; Eq.1; reading A2).
// Shared by the sampler (per-ray F(d), written once into the ray record) and the MLP kernel (F(q)).
#pragma once
#include <cuda_bf16.h>
#include <stdint.h>

namespace r360 {

constexpr int kTcLp = 10, kTcLd = 4;      // the tensor path is specialised to the paper's PE sizes
constexpr int kTcPeP = 3 + 6 * kTcLp;     // 63
constexpr int kTcPeD = 3 + 6 * kTcLd;     // 27

// two fp32 -> packed bf16x2 (lo = first argument = lower K index), round to nearest even
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// same with ReLU fused into the conversion
__device__ __forceinline__ uint32_t pack_bf16_relu(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// two fp32 -> packed binary16 x2 (lo in the lower half), round to nearest even
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// same with ReLU fused into the conversion; out-of-range magnitudes saturate to the largest finite binary16 value
__device__ __forceinline__ uint32_t pack_f16_relu(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.relu.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// operand format of the tensor path: F16 = false bfloat16, true binary16
template <bool F16>
__device__ __forceinline__ uint32_t pack16(float lo, float hi) {
  if constexpr (F16) return pack_f16(lo, hi);
  else return pack_bf16(lo, hi);
}
template <bool F16>
__device__ __forceinline__ uint32_t pack16_relu(float lo, float hi) {
  if constexpr (F16) return pack_f16_relu(lo, hi);
  else return pack_bf16_relu(lo, hi);
}

// packed binary32 pairs (sm_100: add / mul / fma .f32x2 on a 64-bit register pair)
__device__ __forceinline__ uint64_t pack_f32x2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack_f32x2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t add_f32x2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ uint64_t mul_f32x2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ uint64_t fma_f32x2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

// sin and cos on |x| <= 1 (normalised positions, reading A3, and unit direction components) by
// their Taylor polynomials (remainders x^13/13! and x^14/14! are below binary32 resolution).
__device__ __forceinline__ void sincos_unit(float x, float& s, float& c) {
  const float x2 = x * x;
  float ps = fmaf(x2, -2.5052108e-8f, 2.7557319e-6f);     // -1/11!, 1/9!
  ps = fmaf(x2, ps, -1.9841270e-4f);                      // -1/7!
  ps = fmaf(x2, ps, 8.3333333e-3f);                       // 1/5!
  ps = fmaf(x2, ps, -1.6666667e-1f);                      // -1/3!
  s = fmaf(x * x2, ps, x);
  float pc = fmaf(x2, 2.0876757e-9f, -2.7557319e-7f);     // 1/12!, -1/10!
  pc = fmaf(x2, pc, 2.4801587e-5f);                       // 1/8!
  pc = fmaf(x2, pc, -1.3888889e-3f);                      // -1/6!
  pc = fmaf(x2, pc, 4.1666667e-2f);                       // 1/4!
  pc = fmaf(x2, pc, -0.5f);
  c = fmaf(x2, pc, 1.0f);
}

// sin and TWICE the cosine (all cosine coefficients doubled: exact), for the tensor path's recurrence on q = 2 cos
__device__ __forceinline__ void sin_2cos_unit(float x, float& s, float& q) {
  const float x2 = x * x;
  float ps = fmaf(x2, -2.5052108e-8f, 2.7557319e-6f);
  ps = fmaf(x2, ps, -1.9841270e-4f);
  ps = fmaf(x2, ps, 8.3333333e-3f);
  ps = fmaf(x2, ps, -1.6666667e-1f);
  s = fmaf(x * x2, ps, x);
  float pc = fmaf(x2, 2.0f * 2.0876757e-9f, 2.0f * -2.7557319e-7f);
  pc = fmaf(x2, pc, 2.0f * 2.4801587e-5f);
  pc = fmaf(x2, pc, 2.0f * -1.3888889e-3f);
  pc = fmaf(x2, pc, 2.0f * 4.1666667e-2f);
  pc = fmaf(x2, pc, -1.0f);
  q = fmaf(x2, pc, 2.0f);
}
// the same for two arguments at once in a packed pair
__device__ __forceinline__ void sin_2cos_unit2(uint64_t x, uint64_t& s, uint64_t& q) {
#define R360_K2(v) pack_f32x2(v, v)
  const uint64_t x2 = mul_f32x2(x, x);
  uint64_t ps = fma_f32x2(x2, R360_K2(-2.5052108e-8f), R360_K2(2.7557319e-6f));
  ps = fma_f32x2(x2, ps, R360_K2(-1.9841270e-4f));
  ps = fma_f32x2(x2, ps, R360_K2(8.3333333e-3f));
  ps = fma_f32x2(x2, ps, R360_K2(-1.6666667e-1f));
  s = fma_f32x2(mul_f32x2(x, x2), ps, x);
  uint64_t pc = fma_f32x2(x2, R360_K2(2.0f * 2.0876757e-9f), R360_K2(2.0f * -2.7557319e-7f));
  pc = fma_f32x2(x2, pc, R360_K2(2.0f * 2.4801587e-5f));
  pc = fma_f32x2(x2, pc, R360_K2(2.0f * -1.3888889e-3f));
  pc = fma_f32x2(x2, pc, R360_K2(2.0f * 4.1666667e-2f));
  pc = fma_f32x2(x2, pc, R360_K2(-1.0f));
  q = fma_f32x2(x2, pc, R360_K2(2.0f));
#undef R360_K2
}

// sin and cos of two arguments at once in a packed pair
__device__ __forceinline__ void sincos_unit2(uint64_t x, uint64_t& s, uint64_t& c) {
#define R360_K2(v) pack_f32x2(v, v)
  const uint64_t x2 = mul_f32x2(x, x);
  uint64_t ps = fma_f32x2(x2, R360_K2(-2.5052108e-8f), R360_K2(2.7557319e-6f));
  ps = fma_f32x2(x2, ps, R360_K2(-1.9841270e-4f));
  ps = fma_f32x2(x2, ps, R360_K2(8.3333333e-3f));
  ps = fma_f32x2(x2, ps, R360_K2(-1.6666667e-1f));
  s = fma_f32x2(mul_f32x2(x, x2), ps, x);
  uint64_t pc = fma_f32x2(x2, R360_K2(2.0876757e-9f), R360_K2(-2.7557319e-7f));
  pc = fma_f32x2(x2, pc, R360_K2(2.4801587e-5f));
  pc = fma_f32x2(x2, pc, R360_K2(-1.3888889e-3f));
  pc = fma_f32x2(x2, pc, R360_K2(4.1666667e-2f));
  pc = fma_f32x2(x2, pc, R360_K2(-0.5f));
  c = fma_f32x2(x2, pc, R360_K2(1.0f));
#undef R360_K2
}

// F(x) for L levels from one sincos per component and the double-angle recurrence
// (s' = 2 s c, c' = 1 - 2 s^2); out[3 + 6l + a] = sin, out[3 + 6l + 3 + a] = cos (reading A2).
template <int L>
__device__ __forceinline__ void pe_recurrence(const float x[3], float* out) {
  float s[3], c[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    out[a] = x[a];
    sincos_unit(x[a], s[a], c[a]);
  }
#pragma unroll
  for (int l = 0; l < L; ++l) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      out[3 + 6 * l + a] = s[a];
      out[3 + 6 * l + 3 + a] = c[a];
      float t = s[a] + s[a];
      float s2 = t * c[a];
      c[a] = fmaf(-t, s[a], 1.0f);
      s[a] = s2;
    }
  }
}

// Per-ray direction block of the tensor path (64 bytes = 32 values in the operand format): [1, 1, F(d) (27), 0, 0, 0].
// It is the tail of the A operand of every layer after the first: the two ones feed the bias hi/lo
// rows of the hidden layers (first 16 entries = one K step), the whole block feeds the colour layer.
constexpr int kDirBlockWords = 16;

template <bool F16>
__device__ __forceinline__ void store_dir_block(uint4* dst, const float d[3]) {
  float pd[32];
  pd[0] = 1.0f;
  pd[1] = 1.0f;
  pe_recurrence<kTcLd>(d, pd + 2);
#pragma unroll
  for (int c = 2 + kTcPeD; c < 32; ++c) pd[c] = 0.0f;
#pragma unroll
  for (int c = 0; c < 4; ++c)
    dst[c] = make_uint4(pack16<F16>(pd[8 * c], pd[8 * c + 1]), pack16<F16>(pd[8 * c + 2], pd[8 * c + 3]),
                        pack16<F16>(pd[8 * c + 4], pd[8 * c + 5]), pack16<F16>(pd[8 * c + 6], pd[8 * c + 7]));
}

}  // namespace r360
