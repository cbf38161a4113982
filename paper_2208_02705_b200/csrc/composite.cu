// r360 -- per-ray volume compositing with transmittance early-out (step a10).
// Eq.4: C = sum w_i c_i, D = sum w_i t_i; Eq.5 (:96-99): w_i = T_i alpha_i with
// alpha_i = 1 - exp(-sigma_i delta_i); readings E (delta_i = the sample's stratum) and G (running
// product, stop after the first sample with T < tau, black background, depth not normalised).
#include <cuda_fp16.h>

#include "kernels.h"

namespace r360 {

__device__ __forceinline__ float4 unpack_half4(uint2 q) {
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&q.x));
  const float2 c = __half22float2(*reinterpret_cast<const __half2*>(&q.y));
  return make_float4(a.x, a.y, c.x, c.y);
}

__device__ __forceinline__ void write_pixel(const FrameParams& f, void* out_rgb, void* out_depth, size_t gr, float C0,
                                            float C1, float C2, float D) {
  if (f.out_format == 0) {
    float* o = reinterpret_cast<float*>(out_rgb) + gr * 3;
    o[0] = C0; o[1] = C1; o[2] = C2;
    reinterpret_cast<float*>(out_depth)[gr] = D;
  } else {
    // R360_OUT_RGB8_D16: colour rounded to the nearest of 256 levels, depth to binary16
    uint8_t* o = reinterpret_cast<uint8_t*>(out_rgb) + gr * 3;
    o[0] = (uint8_t)__float2int_rn(__saturatef(C0) * 255.0f);
    o[1] = (uint8_t)__float2int_rn(__saturatef(C1) * 255.0f);
    o[2] = (uint8_t)__float2int_rn(__saturatef(C2) * 255.0f);
    reinterpret_cast<__half*>(out_depth)[gr] = __float2half_rn(D);
  }
}

// Tensor path, KK samples of 8 bytes per segment (KK even: whole 16-byte words): the NEXT segment's samples are
// requested before this one's are composited, so two segments are in flight per ray.
template <int KK>
__device__ __forceinline__ void composite_half_segments(const ChunkBuffers& b, unsigned off, unsigned cnt, float tau,
                                                        float& T, float& C0, float& C1, float& C2, float& D,
                                                        unsigned& used, bool& done) {
  constexpr int Q = KK / 2;
  const uint4* o = reinterpret_cast<const uint4*>(reinterpret_cast<const uint2*>(b.out) + (size_t)off * KK);
  uint4 q[Q], qn[Q];
  const float2 td0 = b.seg_td[off];
  float t_in = td0.x, dt = td0.y, t_in_n = 0.f, dt_n = 0.f;
#pragma unroll
  for (int u = 0; u < Q; ++u) q[u] = __ldcs(o + u);
  for (unsigned s = 0; s < cnt && !done; ++s) {
    if (s + 1 < cnt) {
#pragma unroll
      for (int u = 0; u < Q; ++u) qn[u] = __ldcs(o + (size_t)(s + 1) * Q + u);
      const float2 tdn = b.seg_td[off + s + 1];
      t_in_n = tdn.x;
      dt_n = tdn.y;
    }
#pragma unroll
    for (int u = 0; u < KK; ++u) {
      if (!done) {
        const uint4 qq = q[u >> 1];
        const float4 v = unpack_half4((u & 1) ? make_uint2(qq.z, qq.w) : make_uint2(qq.x, qq.y));
        const float t = __fmaf_rn((float)u + 0.5f, dt, t_in);
        const float alpha = 1.0f - expf(-v.x * dt);
        const float w = T * alpha;
        C0 = fmaf(w, v.y, C0);
        C1 = fmaf(w, v.z, C1);
        C2 = fmaf(w, v.w, C2);
        D = fmaf(w, t, D);
        T = T * (1.0f - alpha);
        ++used;
        if (T < tau) done = true;
      }
    }
#pragma unroll
    for (int u = 0; u < Q; ++u) q[u] = qn[u];
    t_in = t_in_n;
    dt = dt_n;
  }
}

// HALF: the tensor path writes a sample as four binary16 values (sigma, r, g, b), 8 bytes
// KFAST: 8 / 12 / 16 = the tensor path's pipelined loop for that K (its own kernel, so that the wider variants'
// registers do not cost the K = 8 case occupancy); 0 = the general loop
template <bool HALF, int KFAST>
__global__ void __launch_bounds__(128)
k_composite(GridParams g, FrameParams f, ChunkBuffers b, float tau, void* __restrict__ out_rgb,
            void* __restrict__ out_depth, PassParams pp) {
  const unsigned r = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned used = 0;
  if (chunk_cancelled(b)) return;
  // wavefront pass: rays that finished in an earlier pass have nothing left to do
  if (r < f.n_rays && !(pp.wavefront && !pp.first && b.st_T[r] < 0.0f)) {
    const unsigned cnt = pp.wavefront ? b.pass_cnt[r] : b.ray_cnt[r];
    const unsigned off = pp.wavefront ? b.pass_off[r] : b.ray_off[r];
    const int K = g.K;
    float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f, D = 0.f;
    if (pp.wavefront && !pp.first) {       // the sums continue exactly where the previous pass left them
      const float4 c = b.st_c[r];
      C0 = c.x; C1 = c.y; C2 = c.z; D = c.w;
      T = b.st_T[r];
    }
    bool done = false;
    unsigned s_begin = 0;
    if constexpr (HALF && KFAST > 0) {
      if (cnt) composite_half_segments<KFAST>(b, off, cnt, tau, T, C0, C1, C2, D, used, done);
      s_begin = cnt;                       // nothing left for the general loop
    }
    for (unsigned s = s_begin; s < cnt && !done; ++s) {
      const float2 td = b.seg_td[off + s];
      const float t_in = td.x, dt = td.y;
      const size_t o0 = (size_t)(off + s) * K;
      // the K samples of a segment are K consecutive float4 (uint2 on the tensor path): fetch them eight at a
      // time, back to back, so that every 128-byte line is requested once, whole, and not re-fetched after an
      // L1 eviction
      for (int j0 = 0; j0 < K && !done; j0 += 8) {
        float4 v[8];
        if constexpr (HALF) {
          const uint2* o = reinterpret_cast<const uint2*>(b.out) + o0;
          if (j0 + 8 <= K && ((o0 + j0) & 1) == 0) {
            uint4 q[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) q[u] = __ldcs(reinterpret_cast<const uint4*>(o + j0) + u);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              v[2 * u] = unpack_half4(make_uint2(q[u].x, q[u].y));
              v[2 * u + 1] = unpack_half4(make_uint2(q[u].z, q[u].w));
            }
          } else {
#pragma unroll
            for (int u = 0; u < 8; ++u)
              if (j0 + u < K) v[u] = unpack_half4(__ldcs(o + j0 + u));
          }
        } else {
          const float4* o = b.out + o0;
#pragma unroll
          for (int u = 0; u < 8; ++u)
            if (j0 + u < K) v[u] = __ldcs(o + j0 + u);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          if (j0 + u < K && !done) {
            const float t = __fmaf_rn((float)(j0 + u) + 0.5f, dt, t_in);
            const float alpha = 1.0f - expf(-v[u].x * dt);
            const float w = T * alpha;
            C0 = fmaf(w, v[u].y, C0);
            C1 = fmaf(w, v[u].z, C1);
            C2 = fmaf(w, v[u].w, C2);
            D = fmaf(w, t, D);
            T = T * (1.0f - alpha);
            ++used;
            if (T < tau) done = true;
          }
        }
      }
    }
    bool write_out = true;
    if (pp.wavefront) {
      // finished: stopped by tau, no hits beyond this pass, or last pass
      const bool finished = done || pp.last || b.ray_cnt[r] <= pp.h1;
      if (!finished) {
        b.st_c[r] = make_float4(C0, C1, C2, D);
        b.st_T[r] = T;
      } else {
        b.st_T[r] = -1.0f;
      }
      write_out = finished;
    }
    if (write_out) {
      write_pixel(f, out_rgb, out_depth, (size_t)(f.out0 + (long long)r), C0, C1, C2, D);
    }
  }
  // samples_used statistic
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) used += __shfl_xor_sync(0xffffffffu, used, o);
  if ((threadIdx.x & 31) == 0 && used) atomicAdd(&b.totals[kTotUsed], (unsigned long long)used);
}

// debug tap: the per-sample MLP outputs (sigma, r, g, b), ray-major, as float4
__global__ void k_export_field(ChunkBuffers b, size_t n_samples, int half_samples, float4* __restrict__ field) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_samples) return;
  field[i] = half_samples ? unpack_half4(reinterpret_cast<const uint2*>(b.out)[i]) : b.out[i];
}

void launch_export_field(const ChunkBuffers& b, size_t n_samples, bool half_samples, float* field, cudaStream_t s) {
  if (!n_samples) return;
  k_export_field<<<(unsigned)((n_samples + 255) / 256), 256, 0, s>>>(b, n_samples, half_samples ? 1 : 0,
                                                                     reinterpret_cast<float4*>(field));
}

void launch_composite(const GridParams& g, const FrameParams& f, const ChunkBuffers& b, float tau,
                      void* out_rgb, void* out_depth, const PassParams& pp, bool half_samples, cudaStream_t s) {
  const dim3 grid((f.n_rays + 127) / 128), block(128);
  if (!half_samples) k_composite<false, 0><<<grid, block, 0, s>>>(g, f, b, tau, out_rgb, out_depth, pp);
  else if (g.K == 8) k_composite<true, 8><<<grid, block, 0, s>>>(g, f, b, tau, out_rgb, out_depth, pp);
  else if (g.K == 12) k_composite<true, 12><<<grid, block, 0, s>>>(g, f, b, tau, out_rgb, out_depth, pp);
  else if (g.K == 16) k_composite<true, 16><<<grid, block, 0, s>>>(g, f, b, tau, out_rgb, out_depth, pp);
  else k_composite<true, 0><<<grid, block, 0, s>>>(g, f, b, tau, out_rgb, out_depth, pp);
}

}  // namespace r360
