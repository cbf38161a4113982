// r360 -- grouped tiny-MLP, fp32 on the FP32 ALUs (steps a6-a9; the 1e-4 parity path).
//
// One CTA = 128 threads = one 128-row tile (128/K segments x K samples) of ONE subfield at a
// time; a CTA owns a contiguous range of tiles, so it re-stages weights only when the subfield
// changes.  Weights sit in shared memory transposed (W^T[in][out]) so the inner loop over the
// outputs reads float4 broadcasts; each thread keeps its row's accumulators in registers and
// its activations in a private shared-memory column (no barrier inside a tile).
// Eq.1, layer layout reading A1, heads A4 (Table 4 :438-442).
#include "kernels.h"

namespace r360 {

template <int WD>
__device__ __forceinline__ void axpy(float (&acc)[WD], const float* __restrict__ wrow, float x) {
#pragma unroll
  for (int o = 0; o < WD; o += 4) {
    float4 w = *reinterpret_cast<const float4*>(wrow + o);
    acc[o + 0] = fmaf(w.x, x, acc[o + 0]);
    acc[o + 1] = fmaf(w.y, x, acc[o + 1]);
    acc[o + 2] = fmaf(w.z, x, acc[o + 2]);
    acc[o + 3] = fmaf(w.w, x, acc[o + 3]);
  }
}

template <int WD>
__device__ __forceinline__ void load_bias(float (&acc)[WD], const float* __restrict__ b) {
#pragma unroll
  for (int o = 0; o < WD; o += 4) {
    float4 w = *reinterpret_cast<const float4*>(b + o);
    acc[o] = w.x; acc[o + 1] = w.y; acc[o + 2] = w.z; acc[o + 3] = w.w;
  }
}

// acc += W^T[row0 .. row0+3+6L) * F(x)   (reading A2: [x, sin 2^l x (xyz), cos 2^l x (xyz), ...])
template <int WD>
__device__ __forceinline__ void pe_axpy(float (&acc)[WD], const float* __restrict__ W, const float x[3], int L) {
#pragma unroll
  for (int a = 0; a < 3; ++a) axpy<WD>(acc, W + a * WD, x[a]);
  float fr = 1.0f;
  for (int l = 0; l < L; ++l) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      float s, c;
      sincosf(fr * x[a], &s, &c);       // 2^l * x is exact
      axpy<WD>(acc, W + (3 + 6 * l + a) * WD, s);
      axpy<WD>(acc, W + (3 + 6 * l + 3 + a) * WD, c);
    }
    fr *= 2.0f;
  }
}

template <int WD>
__global__ void __launch_bounds__(kTileRows)
k_mlp_fp32(GridParams g, FrameParams f, ChunkBuffers b, NetShape net, Fp32Layout lay,
           const float* __restrict__ wt, const SubfieldFrame* __restrict__ frames, int n_bins, int spt) {
  extern __shared__ __align__(16) float smem[];
  float* sw = smem;                       // [lay.total]
  float* act = smem + lay.total;          // [WD][128], column = thread
  const int tid = threadIdx.x;
  if (chunk_cancelled(b)) return;
  const unsigned total_tiles = (unsigned)b.totals[kTotTiles];
  const unsigned per = (total_tiles + gridDim.x - 1) / gridDim.x;
  const unsigned tile0 = blockIdx.x * per;
  const unsigned tile1 = min(total_tiles, tile0 + per);
  int cur_k = -1;
  const int K = g.K;
  for (unsigned tile = tile0; tile < tile1; ++tile) {
    // subfield of this tile: last k with tile_start[k] <= tile
    int lo = 0, hi = n_bins;
    while (hi - lo > 1) {
      int mid = (lo + hi) >> 1;
      if (__ldg(b.tile_start + mid) <= tile) lo = mid; else hi = mid;
    }
    const int k = lo;
    if (k != cur_k) {
      __syncthreads();
      const float4* src = reinterpret_cast<const float4*>(wt + (size_t)k * lay.total);
      float4* dst = reinterpret_cast<float4*>(sw);
      for (int i = tid; i < lay.total / 4; i += kTileRows) dst[i] = __ldg(src + i);
      __syncthreads();
      cur_k = k;
    }
    const unsigned seg0 = __ldg(b.bin_start + k) + (tile - __ldg(b.tile_start + k)) * spt;
    const unsigned nseg = min((unsigned)spt, __ldg(b.bin_start + k + 1) - seg0);
    const int sidx = tid / K, j = tid - sidx * K;
    const bool active = (unsigned)sidx < nseg;
    SegRec rec = make_uint4(0, 0, 0, 0);
    if (active) rec = b.recs[(size_t)(seg0 + sidx) * kRecWords];
    const float t_in = __uint_as_float(rec.y), dt = __uint_as_float(rec.z);
    const float t = __fmaf_rn((float)j + 0.5f, dt, t_in);            // reading D
    const Ray ray = make_ray(f, active ? rec.x : 0u);
    const SubfieldFrame fr = frames[k];
    float q[3];                                                       // reading A3
    q[0] = __fmul_rn(__fsub_rn(__fmaf_rn(t, ray.d[0], ray.o[0]), fr.cx), fr.ix);
    q[1] = __fmul_rn(__fsub_rn(__fmaf_rn(t, ray.d[1], ray.o[1]), fr.cy), fr.iy);
    q[2] = __fmul_rn(__fsub_rn(__fmaf_rn(t, ray.d[2], ray.o[2]), fr.cz), fr.iz);

    float acc[WD];
    // trunk-1
    {
      const float* W = sw + lay.trunk[0];
      load_bias<WD>(acc, W + net.pe_p * WD);
      pe_axpy<WD>(acc, W, q, net.Lp);
#pragma unroll
      for (int o = 0; o < WD; ++o) act[o * kTileRows + tid] = fmaxf(acc[o], 0.0f);
    }
    // trunk-2..Hd
    for (int l = 1; l < net.Hd; ++l) {
      const float* W = sw + lay.trunk[l];
      load_bias<WD>(acc, W + WD * WD);
#pragma unroll 4
      for (int i = 0; i < WD; ++i) axpy<WD>(acc, W + i * WD, act[i * kTileRows + tid]);
#pragma unroll
      for (int o = 0; o < WD; ++o) act[o * kTileRows + tid] = fmaxf(acc[o], 0.0f);
    }
    // density head
    float sigma_raw;
    {
      const float* W = sw + lay.dens;
      sigma_raw = W[WD];
#pragma unroll 8
      for (int i = 0; i < WD; ++i) sigma_raw = fmaf(W[i], act[i * kTileRows + tid], sigma_raw);
    }
    // feature (no activation)
    {
      const float* W = sw + lay.feat;
      load_bias<WD>(acc, W + WD * WD);
#pragma unroll 4
      for (int i = 0; i < WD; ++i) axpy<WD>(acc, W + i * WD, act[i * kTileRows + tid]);
#pragma unroll
      for (int o = 0; o < WD; ++o) act[o * kTileRows + tid] = acc[o];
    }
    // colour layer on [feature, F(d)], ReLU
    {
      const float* W = sw + lay.col;
      load_bias<WD>(acc, W + (WD + net.pe_d) * WD);
#pragma unroll 4
      for (int i = 0; i < WD; ++i) axpy<WD>(acc, W + i * WD, act[i * kTileRows + tid]);
      pe_axpy<WD>(acc, W + WD * WD, ray.d, net.Ld);
    }
    // rgb
    float c0, c1, c2;
    {
      const float* W = sw + lay.rgb;
      c0 = W[WD * 4 + 0]; c1 = W[WD * 4 + 1]; c2 = W[WD * 4 + 2];
#pragma unroll
      for (int i = 0; i < WD; ++i) {
        float x = fmaxf(acc[i], 0.0f);
        float4 w = *reinterpret_cast<const float4*>(W + i * 4);
        c0 = fmaf(w.x, x, c0); c1 = fmaf(w.y, x, c1); c2 = fmaf(w.z, x, c2);
      }
    }
    // heads (A4)
    float sigma = net.act == 1 ? (sigma_raw > 20.0f ? sigma_raw : log1pf(expf(sigma_raw)))
                               : fmaxf(sigma_raw, 0.0f);
    float4 o4;
    o4.x = sigma;
    o4.y = 1.0f / (1.0f + expf(-c0));
    o4.z = 1.0f / (1.0f + expf(-c1));
    o4.w = 1.0f / (1.0f + expf(-c2));
    if (active) b.out[(size_t)rec.w * K + j] = o4;
  }
}

template <int WD>
static cudaError_t launch_t(const GridParams& g, const FrameParams& f, const ChunkBuffers& b, const NetShape& net,
                            const Fp32Layout& lay, const float* wt, const SubfieldFrame* frames, int n_bins,
                            int spt, int n_sms, cudaStream_t s) {
  size_t smem = ((size_t)lay.total + (size_t)WD * kTileRows) * sizeof(float);
  cudaError_t e = cudaFuncSetAttribute(k_mlp_fp32<WD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int per_sm = 1;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_mlp_fp32<WD>, kTileRows, smem);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) per_sm = 1;
  k_mlp_fp32<WD><<<n_sms * per_sm, kTileRows, smem, s>>>(g, f, b, net, lay, wt, frames, n_bins, spt);
  return cudaGetLastError();
}

cudaError_t launch_mlp_fp32(const GridParams& g, const FrameParams& f, const ChunkBuffers& b,
                            const NetShape& net, const Fp32Layout& lay, const float* weights_t,
                            const SubfieldFrame* frames, int n_bins, int segs_per_tile, int n_sms,
                            cudaStream_t s) {
  if (net.Wd == 32) return launch_t<32>(g, f, b, net, lay, weights_t, frames, n_bins, segs_per_tile, n_sms, s);
  if (net.Wd == 64) return launch_t<64>(g, f, b, net, lay, weights_t, frames, n_bins, segs_per_tile, n_sms, s);
  return cudaErrorInvalidValue;
}

}  // namespace r360
