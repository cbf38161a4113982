// r360 -- grouped tiny-MLP on the 5th-gen tensor cores (steps a6-a9, bf16 operands, fp32 accumulate).
//
// One CTA = 128 threads = one 128-row tile (128/K segments x K samples) of one subfield at a time;
// thread r owns sample row r end to end.  Every layer is D[128 x N] = A[128 x Kpad] * B[N x Kpad]^T:
//   A  lives in TENSOR MEMORY: the owning thread writes its row (bf16x2-packed) with tcgen05.st, so
//      activations never touch shared memory and the MMA reads only B (the weights) from SMEM;
//   B  = the subfield's weights, pre-packed on the host into the UMMA K-major no-swizzle core-matrix
//      layout and staged with ONE TMA bulk copy per subfield change;
//   D  accumulates in TMEM and comes back with tcgen05.ld for the bias-free epilogue:
//      biases ride in the GEMM as two extra K rows (hi + lo bf16 parts) against constant-1 inputs,
//      so the epilogue per element is one cvt.rn.relu.bf16x2 per pair.
// One thread issues the tcgen05.mma's of a layer and commits them to an mbarrier; latency of the
// st -> mma -> ld chain is hidden by running several CTAs per SM (TMEM: 128/256 columns per CTA).
// Eq.1, layer layout reading A1, heads A4 (Table 4 :438-442).
#include <cstring>
#include <vector>

#include "kernels.h"
#include "tc_ptx.cuh"

namespace r360 {

namespace {

constexpr int kLp = 10, kLd = 4;          // the tensor path is specialised to the paper's PE sizes
constexpr int kPeP = 3 + 6 * kLp;         // 63
constexpr int kPeD = 3 + 6 * kLd;         // 27

template <int WD>
struct TcShape {
  static constexpr int KP1 = 64;                          // trunk-1 inputs: 63 -> 64
  static constexpr int ND = WD + 16;                      // density+feature outputs: WD+1 -> WD+16
  static constexpr int KC = ((WD + kPeD + 2 + 15) / 16) * 16;  // colour inputs [feature, F(d), 1, 1] -> 64 / 96
  static constexpr int NRGB = 16;                         // rgb outputs: 3 -> 16
  // TMEM columns
  static constexpr int D_COL = 0;                         // accumulator, up to ND columns
  static constexpr int A_COL = ND;                        // A operand, up to max(KP1, KC)/2 columns
  static constexpr int A_COLS = (KP1 > KC ? KP1 : KC) / 2;
  static constexpr int ONE_COL = A_COL + A_COLS;          // constant-1 block (8 columns)
  static constexpr int TMEM_COLS = (ONE_COL + 8) <= 128 ? 128 : 256;
  static constexpr int CTAS_PER_SM = 512 / TMEM_COLS;
  // bytes of one K=16 step of a B operand with N rows
  __host__ __device__ static constexpr int blk(int N) { return N * 32; }
};

// byte offsets of the layers inside one subfield's packed blob
struct TcLayout {
  int trunk[8];
  int df, col, rgb, total;
};

template <int WD>
TcLayout make_tc_layout(int Hd) {
  using S = TcShape<WD>;
  TcLayout L{};
  int o = 0;
  L.trunk[0] = o; o += (S::KP1 / 16 + 1) * S::blk(WD);
  for (int l = 1; l < Hd; ++l) { L.trunk[l] = o; o += (WD / 16 + 1) * S::blk(WD); }
  L.df = o; o += (WD / 16 + 1) * S::blk(S::ND);
  L.col = o; o += (S::KC / 16) * S::blk(WD);
  L.rgb = o; o += (WD / 16 + 1) * S::blk(S::NRGB);
  L.total = o;
  return L;
}

uint16_t bf16_bits(float f) {            // round to nearest even (finite inputs)
  uint32_t u;
  std::memcpy(&u, &f, 4);
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
float bf16_value(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  std::memcpy(&f, &u, 4);
  return f;
}

// element (n, k) of a B operand with N rows -> halfword index inside the layer's packed bytes
inline size_t b_index(int N, int n, int k) {
  int s = k / 16, c = (k % 16) / 8, e = k % 8, g = n / 8, r = n % 8;
  return (size_t)s * N * 16 + (size_t)g * 128 + c * 64 + r * 8 + e;
}

// pack one layer: rows n < n_out come from W[n][k_src] (k < k_in) and bias b[n] (hi at k_bias, lo at
// k_bias+1); everything else is zero.
void pack_layer(uint16_t* dst, int N, const float* W, const float* b, int n_out, int k_in, int k_bias) {
  for (int n = 0; n < n_out; ++n) {
    for (int k = 0; k < k_in; ++k) dst[b_index(N, n, k)] = bf16_bits(W[(size_t)n * k_in + k]);
    uint16_t hi = bf16_bits(b[n]);
    dst[b_index(N, n, k_bias)] = hi;
    dst[b_index(N, n, k_bias + 1)] = bf16_bits(b[n] - bf16_value(hi));
  }
}

template <int WD>
void pack_subfield_t(const NetShape& net, const float* src, void* dstv) {
  using S = TcShape<WD>;
  TcLayout L = make_tc_layout<WD>(net.Hd);
  std::memset(dstv, 0, (size_t)L.total);
  unsigned char* dst = (unsigned char*)dstv;
  const float* s = src;
  // trunk-1: W[WD][63], bias rows at k = 64, 65 (the extra K=16 block)
  pack_layer((uint16_t*)(dst + L.trunk[0]), WD, s, s + WD * kPeP, WD, kPeP, S::KP1);
  s += WD * kPeP + WD;
  for (int l = 1; l < net.Hd; ++l) {
    pack_layer((uint16_t*)(dst + L.trunk[l]), WD, s, s + WD * WD, WD, WD, WD);
    s += WD * WD + WD;
  }
  // density (row WD) + feature (rows 0..WD-1), N = ND
  const float* dens = s; s += WD + 1;
  const float* feat = s; s += WD * WD + WD;
  pack_layer((uint16_t*)(dst + L.df), S::ND, feat, feat + WD * WD, WD, WD, WD);
  {
    uint16_t* d = (uint16_t*)(dst + L.df);
    for (int k = 0; k < WD; ++k) d[b_index(S::ND, WD, k)] = bf16_bits(dens[k]);
    uint16_t hi = bf16_bits(dens[WD]);
    d[b_index(S::ND, WD, WD)] = hi;
    d[b_index(S::ND, WD, WD + 1)] = bf16_bits(dens[WD] - bf16_value(hi));
  }
  // colour: inputs [feature(WD), F(d)(27)], bias at the two spare slots WD+27, WD+28
  pack_layer((uint16_t*)(dst + L.col), WD, s, s + WD * (WD + kPeD), WD, WD + kPeD, WD + kPeD);
  s += WD * (WD + kPeD) + WD;
  pack_layer((uint16_t*)(dst + L.rgb), S::NRGB, s, s + 3 * WD, 3, WD, WD);
}

}  // namespace

size_t tc_pack_stride(const NetShape& net) {
  if (net.Lp != kLp || net.Ld != kLd) return 0;      // tensor path: paper's PE sizes only
  if (net.Wd == 32) return (size_t)make_tc_layout<32>(net.Hd).total;
  if (net.Wd == 64) return (size_t)make_tc_layout<64>(net.Hd).total;
  return 0;
}

void tc_pack_subfield(const NetShape& net, const float* src_blob, void* dst) {
  if (net.Wd == 32) pack_subfield_t<32>(net, src_blob, dst);
  else if (net.Wd == 64) pack_subfield_t<64>(net, src_blob, dst);
}

// ---------------------------------------------------------------------------------------------
using namespace tc;

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

// heads of the bf16 path: ex2/lg2/rcp approximations (relative error ~2^-22, far below bf16)
__device__ __forceinline__ float fast_sigmoid(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + __expf(-x)));
  return r;
}
__device__ __forceinline__ float fast_softplus(float x) {
  return x > 20.0f ? x : __logf(1.0f + __expf(x));
}

template <int WD>
__global__ void __launch_bounds__(kTileRows, TcShape<WD>::CTAS_PER_SM)
k_mlp_tc(GridParams g, FrameParams f, ChunkBuffers b, NetShape net, TcLayout lay,
         const unsigned char* __restrict__ wpack, const SubfieldFrame* __restrict__ frames, int n_bins,
         int spt) {
  using S = TcShape<WD>;
  extern __shared__ __align__(128) unsigned char sw[];      // packed weights of the current subfield
  __shared__ __align__(8) uint64_t bar_w, bar_d;
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, warp = tid >> 5;
  const unsigned total_tiles = (unsigned)b.totals[1];
  const unsigned per = (total_tiles + gridDim.x - 1) / gridDim.x;
  const unsigned tile0 = blockIdx.x * per;
  const unsigned tile1 = min(total_tiles, tile0 + per);
  if (tile0 >= tile1) return;                                // uniform: nothing allocated yet

  if (tid == 0) {
    mbar_init(&bar_w, 1);
    mbar_init(&bar_d, 1);
    mbar_fence_init();
  }
  if (warp == 0) tmem_alloc<S::TMEM_COLS>(&tmem_base_s);
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tbase = tmem_base_s;
  const uint32_t lane_base = tbase + ((uint32_t)(warp * 32) << 16);
  const uint32_t tD = lane_base + S::D_COL, tA = lane_base + S::A_COL;
  {  // constant-1 block: k = 0, 1 are 1.0 (bias hi / lo rows), the rest 0
    uint32_t ones[8] = {0x3F803F80u, 0, 0, 0, 0, 0, 0, 0};
    tmem_st_x8(lane_base + S::ONE_COL, ones);
  }
  const uint32_t sw_addr = smem_u32(sw);
  const uint32_t idesc_w = instr_desc_bf16(128, WD), idesc_d = instr_desc_bf16(128, S::ND),
                 idesc_r = instr_desc_bf16(128, S::NRGB);
  uint32_t par_d = 0, par_w = 0;
  int cur_k = -1;
  const int K = g.K;

  // one layer's MMAs: KS data steps over A, then (bias_block) one step over the constant-1 block
  auto issue = [&](int b_off, int N, uint32_t idesc, int ks_data, bool bias_block) {
    fence_after_sync();
    for (int s = 0; s < ks_data; ++s)
      mma_ts(tbase + S::D_COL, tbase + S::A_COL + 8 * s, smem_desc(sw_addr + b_off + s * S::blk(N), 128, 256),
             idesc, s > 0);
    if (bias_block)
      mma_ts(tbase + S::D_COL, tbase + S::ONE_COL, smem_desc(sw_addr + b_off + ks_data * S::blk(N), 128, 256),
             idesc, 1);
    mma_commit(&bar_d);
  };
  // publish this thread's A row, let one thread issue, wait for the accumulator
  auto run_layer = [&](int b_off, int N, uint32_t idesc, int ks_data, bool bias_block) {
    wait_st();
    fence_before_sync();
    __syncthreads();
    if (tid == 0) issue(b_off, N, idesc, ks_data, bias_block);
  };
  auto wait_acc = [&]() {
    mbar_wait(&bar_d, par_d);
    par_d ^= 1;
    fence_after_sync();
  };
  // D[0..WD) -> (ReLU) -> bf16x2 -> A[0..WD/2)
  auto d_to_a = [&](bool relu) {
    uint32_t d[WD];
#pragma unroll
    for (int c = 0; c < WD; c += 16) tmem_ld_x16(tD + c, d + c);
    wait_ld();
    uint32_t a[WD / 2];
#pragma unroll
    for (int c = 0; c < WD / 2; ++c)
      a[c] = relu ? pack_bf16_relu(__uint_as_float(d[2 * c]), __uint_as_float(d[2 * c + 1]))
                  : pack_bf16(__uint_as_float(d[2 * c]), __uint_as_float(d[2 * c + 1]));
#pragma unroll
    for (int c = 0; c < WD / 2; c += 16) tmem_st_x16(tA + c, a + c);
  };

  unsigned k_tile_end = 0, k_tile_begin = 0, k_seg_begin = 0, k_seg_end = 0;
  SubfieldFrame fr = frames[0];
  for (unsigned tile = tile0; tile < tile1; ++tile) {
    if (tile >= k_tile_end || cur_k < 0) {
      // subfield of this tile: last k with tile_start[k] <= tile (tiles of a CTA are contiguous, so
      // this search runs once per subfield, not once per tile)
      int lo = 0, hi = n_bins;
      while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(b.tile_start + mid) <= tile) lo = mid; else hi = mid;
      }
      const int k = lo;
      k_tile_begin = __ldg(b.tile_start + k);
      k_tile_end = __ldg(b.tile_start + k + 1);
      k_seg_begin = __ldg(b.bin_start + k);
      k_seg_end = __ldg(b.bin_start + k + 1);
      fr = frames[k];
      // stage the subfield's weights (TMA bulk copy)
      __syncthreads();                                       // every MMA reading the old weights has completed
      if (tid == 0) {
        mbar_expect_tx(&bar_w, (uint32_t)lay.total);
        bulk_g2s(sw, wpack + (size_t)k * lay.total, (uint32_t)lay.total, &bar_w);
      }
      cur_k = k;
      mbar_wait(&bar_w, par_w);
      par_w ^= 1;
    }
    const unsigned seg0 = k_seg_begin + (tile - k_tile_begin) * spt;
    const unsigned nseg = min((unsigned)spt, k_seg_end - seg0);
    const int sidx = tid / K, j = tid - sidx * K;
    const bool active = (unsigned)sidx < nseg;
    SegRec rec = make_uint4(0, 0, 0, 0);
    if (active) rec = b.recs[seg0 + sidx];
    const float t_in = __uint_as_float(rec.y), dt = __uint_as_float(rec.z);
    const float t = __fmaf_rn((float)j + 0.5f, dt, t_in);
    const Ray ray = make_ray(f, active ? rec.x : 0u);
    float q[3];
    q[0] = __fmul_rn(__fsub_rn(__fmaf_rn(t, ray.d[0], ray.o[0]), fr.cx), fr.ix);
    q[1] = __fmul_rn(__fsub_rn(__fmaf_rn(t, ray.d[1], ray.o[1]), fr.cy), fr.iy);
    q[2] = __fmul_rn(__fsub_rn(__fmaf_rn(t, ray.d[2], ray.o[2]), fr.cz), fr.iz);

    // ---- trunk-1: A = F(q) (63 values, slot 63 zero), bias block
    {
      float pe[S::KP1];
      pe_recurrence<kLp>(q, pe);
      pe[S::KP1 - 1] = 0.0f;
      uint32_t a[S::KP1 / 2];
#pragma unroll
      for (int c = 0; c < S::KP1 / 2; ++c) a[c] = pack_bf16(pe[2 * c], pe[2 * c + 1]);
#pragma unroll
      for (int c = 0; c < S::KP1 / 2; c += 16) tmem_st_x16(tA + c, a + c);
    }
    run_layer(lay.trunk[0], WD, idesc_w, S::KP1 / 16, true);
    // while the tensor core works: F(d) with the two constant-1 bias slots, packed for the colour layer
    uint32_t ad[(S::KC - WD) / 2];
    {
      float pd[S::KC - WD];
      pe_recurrence<kLd>(ray.d, pd);
      pd[kPeD] = 1.0f;
      pd[kPeD + 1] = 1.0f;
#pragma unroll
      for (int c = kPeD + 2; c < S::KC - WD; ++c) pd[c] = 0.0f;
#pragma unroll
      for (int c = 0; c < (S::KC - WD) / 2; ++c) ad[c] = pack_bf16(pd[2 * c], pd[2 * c + 1]);
    }
    wait_acc();
    // ---- trunk-2..Hd
    for (int l = 1; l < net.Hd; ++l) {
      d_to_a(true);
      if (l == 1) tmem_st_x16(tA + WD / 2, ad);              // F(d) block parks beside the hidden A columns
      run_layer(lay.trunk[l], WD, idesc_w, WD / 16, true);
      wait_acc();
    }
    // ---- density + feature (N = WD+16: columns [0,WD) feature, column WD raw density)
    d_to_a(true);
    if (net.Hd == 1) tmem_st_x16(tA + WD / 2, ad);
    run_layer(lay.df, S::ND, idesc_d, WD / 16, true);
    wait_acc();
    uint32_t sraw[4];
    tmem_ld_x4(tD + WD, sraw);
    // ---- colour layer on [feature, F(d), 1, 1]: feature has no activation; bias in the spare K slots
    d_to_a(false);
    run_layer(lay.col, WD, idesc_w, S::KC / 16, false);
    wait_acc();
    // ---- rgb (N = 16, 3 used)
    d_to_a(true);
    run_layer(lay.rgb, S::NRGB, idesc_r, WD / 16, true);
    wait_acc();
    uint32_t craw[4];
    tmem_ld_x4(tD, craw);
    wait_ld();
    // ---- heads (A4), fp32
    const float sigma_raw = __uint_as_float(sraw[0]);
    float4 o4;
    o4.x = net.act == 1 ? fast_softplus(sigma_raw) : fmaxf(sigma_raw, 0.0f);
    o4.y = fast_sigmoid(__uint_as_float(craw[0]));
    o4.z = fast_sigmoid(__uint_as_float(craw[1]));
    o4.w = fast_sigmoid(__uint_as_float(craw[2]));
    if (active) b.out[(size_t)rec.w * K + j] = o4;
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 0) tmem_dealloc<S::TMEM_COLS>(tbase);
}

template <int WD>
static cudaError_t launch_tc_t(const GridParams& g, const FrameParams& f, const ChunkBuffers& b,
                               const NetShape& net, const void* wpack, const SubfieldFrame* frames, int n_bins,
                               int spt, int n_sms, cudaStream_t s) {
  using S = TcShape<WD>;
  TcLayout lay = make_tc_layout<WD>(net.Hd);
  // shared memory request also caps residency at CTAS_PER_SM so that every CTA owns its TMEM columns
  size_t cap = (size_t)(227 * 1024) / S::CTAS_PER_SM - 2048;
  size_t floor_ = (size_t)(228 * 1024) / (S::CTAS_PER_SM + 1);
  size_t smem = (size_t)lay.total > floor_ ? (size_t)lay.total : floor_;
  if (smem > cap) return cudaErrorInvalidValue;
  cudaError_t e = cudaFuncSetAttribute(k_mlp_tc<WD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_mlp_tc<WD><<<n_sms * S::CTAS_PER_SM, kTileRows, smem, s>>>(g, f, b, net, lay, (const unsigned char*)wpack,
                                                                frames, n_bins, spt);
  return cudaGetLastError();
}

cudaError_t launch_mlp_tc(const GridParams& g, const FrameParams& f, const ChunkBuffers& b, const NetShape& net,
                          const void* wpack, size_t wpack_stride, const SubfieldFrame* frames, int n_bins,
                          int segs_per_tile, int n_sms, cudaStream_t s) {
  if (!wpack || wpack_stride == 0) return cudaErrorNotSupported;
  if (net.Wd == 32) return launch_tc_t<32>(g, f, b, net, wpack, frames, n_bins, segs_per_tile, n_sms, s);
  if (net.Wd == 64) return launch_tc_t<64>(g, f, b, net, wpack, frames, n_bins, segs_per_tile, n_sms, s);
  return cudaErrorInvalidValue;
}

}  // namespace r360
