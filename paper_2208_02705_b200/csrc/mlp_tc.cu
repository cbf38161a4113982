// r360 -- grouped tiny-MLP on the 5th-gen tensor cores (steps a6-a9, bf16 operands, fp32 accumulate).
//
// One CTA per SM holds kGroups independent 128-thread TILE GROUPS (8 for Wd=32, 4 for Wd=64: as many
// as tensor memory allows).  A group works through a contiguous range of 128-row tiles (128/K
// segments x K samples of one subfield); thread r owns sample row r end to end.  Every layer is
// D[128 x N] = A[128 x Kpad] * B[N x Kpad]^T:
//   A  lives in TENSOR MEMORY: the owning thread writes its row (bf16x2-packed) with tcgen05.st, so
//      activations never touch shared memory and the MMA reads only B (the weights) from SMEM;
//   B  = the subfield's weights, pre-packed on the host into the UMMA K-major no-swizzle core-matrix
//      layout and staged with ONE TMA bulk copy per subfield change (one buffer per group);
//   D  accumulates in TMEM and comes back with tcgen05.ld; the epilogue per element pair is one
//      cvt.rn.relu.bf16x2, because the biases ride in the GEMM: the A row of every layer after the
//      first ends with the ray's direction block [1, 1, F(d), 0, 0, 0] (written once per ray by the
//      sampler), whose two ones meet the bias hi/lo rows of B.
// The network evaluated is algebraically the paper's (Eq.1, Table 4 as corrected by PAPER.md:413):
// the feature layer has no activation (Table 4 :439), so it is folded into the colour layer on the
// host (W' = Wc[:, :Wd] Wf, b' = bc + Wc[:, :Wd] bf); the density row then reads the last trunk
// activation directly and is issued together with the rgb layer.  5 dependent layers instead of 6.
// Tensor memory per group (columns): [h : Wd/2 | direction block, later the colour activation :
// max(16, Wd/2) | accumulator : Wd] = 64 (Wd=32) / 128 (Wd=64); all 512 columns are in use.
// One thread per group issues the tcgen05.mma's of a layer and commits them to the group's mbarrier;
// groups synchronise with named barriers only, so the st -> mma -> ld chains of all groups overlap.
// Heads: reading A4 (Table 4 :438-442), biases of the two head rows added in fp32.
#include <cmath>
#include <cstring>
#include <type_traits>
#include <vector>

#include "kernels.h"
#include "tc_ptx.cuh"

namespace r360 {

namespace {

constexpr int kLp = kTcLp, kLd = kTcLd;   // the tensor path is specialised to the paper's PE sizes
constexpr int kPeP = kTcPeP;              // 63
constexpr int kPeD = kTcPeD;              // 27

template <int WD>
struct TcShape {
  static constexpr int KP1 = 64;                          // trunk-1 inputs: F(q) 63 + constant 1 (bias)
  static constexpr int KH = WD + 16;                      // hidden inputs: h + [1, 1, ...] (bias hi/lo)
  static constexpr int KC = WD + 32;                      // colour inputs: h + [1, 1, F(d) 27, 0 0 0]
  static constexpr int NHEAD = 16;                        // rgb (3 used) and density (1 used) outputs
  // TMEM columns of one group
  static constexpr int A_H = 0;                           // h: WD bf16
  static constexpr int A_FD = WD / 2;                     // direction block (16 cols); later colour activation
  static constexpr int D0 = WD / 2 + (WD / 2 > 16 ? WD / 2 : 16);
  static constexpr int G_COLS = D0 + WD;                  // 64 / 128
  static constexpr int kGroups = 512 / G_COLS;            // 8 / 4
  static_assert(KP1 / 2 <= D0, "trunk-1 A operand must fit in front of the accumulator");
  // bytes of one K=16 step of a B operand with N rows
  __host__ __device__ static constexpr int blk(int N) { return N * 32; }
};

// byte offsets of the layers inside one subfield's packed blob
struct TcLayout {
  int trunk[8];
  int col, rgb, dens, head_bias, total;
};

template <int WD>
TcLayout make_tc_layout(int Hd) {
  using S = TcShape<WD>;
  TcLayout L{};
  int o = 0;
  L.trunk[0] = o; o += (S::KP1 / 16) * S::blk(WD);
  for (int l = 1; l < Hd; ++l) { L.trunk[l] = o; o += (S::KH / 16) * S::blk(WD); }
  L.col = o; o += (S::KC / 16) * S::blk(WD);
  L.rgb = o; o += (WD / 16) * S::blk(S::NHEAD);
  L.dens = o; o += (WD / 16) * S::blk(S::NHEAD);
  L.head_bias = o; o += 16;                               // fp32: b_r, b_g, b_b, b_sigma
  L.total = (o + 127) / 128 * 128;
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
// binary16: round to nearest even, subnormals kept, magnitudes beyond the largest finite value saturate to it
// (tc_pack_subfield reports them, and r360_set_precision then refuses the binary16 mode)
constexpr float kF16Max = 65504.0f;
uint16_t f16_bits(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  const uint16_t sign = (uint16_t)((u >> 16) & 0x8000u);
  const float a = std::fabs(f);
  if (!(a <= kF16Max)) return (uint16_t)(sign | 0x7BFFu);
  if (a < 6.103515625e-05f) {              // below 2^-14: a multiple of 2^-24, rounded to nearest even
    const float q = a * 16777216.0f;       // exact scaling
    const float r = std::nearbyint(q);     // default rounding mode: nearest even
    return (uint16_t)(sign | (uint16_t)r);
  }
  uint32_t m = u & 0x7FFFFFFFu;
  m += 0xFFFu + ((m >> 13) & 1u);          // round the 13 dropped mantissa bits to nearest even
  const uint32_t h = ((m >> 13) - (112u << 10));
  return (uint16_t)(sign | (h > 0x7BFFu ? 0x7BFFu : h));
}
float f16_value(uint16_t h) {
  const uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
  const uint32_t e = (h >> 10) & 31u, m = h & 0x3FFu;
  float v;
  if (e == 0) {
    v = (float)m * 5.9604644775390625e-08f;   // 2^-24
  } else {
    const uint32_t u = ((e + 112u) << 23) | (m << 13);
    std::memcpy(&v, &u, 4);
  }
  uint32_t u;
  std::memcpy(&u, &v, 4);
  u |= sign;
  std::memcpy(&v, &u, 4);
  return v;
}

// operand format of one packing run (0 = bfloat16, 1 = binary16) and whether a value left binary16's range
struct PackFmt {
  int f16;
  bool overflow;
  uint16_t bits(float v) {
    if (!f16) return bf16_bits(v);
    if (std::fabs(v) > kF16Max) overflow = true;
    return f16_bits(v);
  }
  float value(uint16_t b) const { return f16 ? f16_value(b) : bf16_value(b); }
};

// element (n, k) of a B operand with N rows -> halfword index inside the layer's packed bytes
inline size_t b_index(int N, int n, int k) {
  int s = k / 16, c = (k % 16) / 8, e = k % 8, g = n / 8, r = n % 8;
  return (size_t)s * N * 16 + (size_t)g * 128 + c * 64 + r * 8 + e;
}
template <int WD>
void pack_subfield_t(const NetShape& net, const float* src, void* dstv, PackFmt& fmt) {
  using S = TcShape<WD>;
  auto put = [&fmt](uint16_t* dst, int N, int n, int k, float v) { dst[b_index(N, n, k)] = fmt.bits(v); };
  auto put_hi_lo = [&fmt](uint16_t* dst, int N, int n, int k, float v) {
    const uint16_t hi = fmt.bits(v);
    dst[b_index(N, n, k)] = hi;
    dst[b_index(N, n, k + 1)] = fmt.bits(v - fmt.value(hi));
  };
  TcLayout L = make_tc_layout<WD>(net.Hd);
  std::memset(dstv, 0, (size_t)L.total);
  unsigned char* dst = (unsigned char*)dstv;
  const float* s = src;
  // trunk-1: W[WD][63]; the bias meets the constant 1 in A slot 63 (one bf16: K is full)
  {
    uint16_t* d = (uint16_t*)(dst + L.trunk[0]);
    const float* W = s; const float* b = s + WD * kPeP;
    for (int n = 0; n < WD; ++n) {
      // cosine columns (k = 3 + 6 l + 3 + a) are halved: the kernel's A row holds 2 cos (store_pe_row)
      for (int k = 0; k < kPeP; ++k) put(d, WD, n, k, (k >= 3 && (k - 3) % 6 >= 3) ? 0.5f * W[n * kPeP + k] : W[n * kPeP + k]);
      put(d, WD, n, kPeP, b[n]);
    }
    s += WD * kPeP + WD;
  }
  // trunk-2..Hd: W[WD][WD]; bias hi/lo against the two ones that open the direction block
  for (int l = 1; l < net.Hd; ++l) {
    uint16_t* d = (uint16_t*)(dst + L.trunk[l]);
    const float* W = s; const float* b = s + WD * WD;
    for (int n = 0; n < WD; ++n) {
      for (int k = 0; k < WD; ++k) put(d, WD, n, k, W[n * WD + k]);
      put_hi_lo(d, WD, n, WD, b[n]);
    }
    s += WD * WD + WD;
  }
  const float* dens = s; s += WD + 1;                     // w[WD], b
  const float* feat = s; s += WD * WD + WD;               // Wf[WD][WD], bf[WD]
  const float* col = s; s += WD * (WD + kPeD) + WD;       // Wc[WD][WD+27] on [feature, F(d)], bc[WD]
  const float* rgb = s;                                   // Wr[3][WD], br[3]
  // colour with the feature layer folded in (no activation between them, Table 4 :439):
  //   pre = (Wc1 Wf) h + Wc2 F(d) + (bc + Wc1 bf), products accumulated in binary64
  {
    uint16_t* d = (uint16_t*)(dst + L.col);
    const float* bc = col + WD * (WD + kPeD);
    for (int n = 0; n < WD; ++n) {
      const float* wc = col + (size_t)n * (WD + kPeD);
      for (int k = 0; k < WD; ++k) {
        double a = 0.0;
        for (int m = 0; m < WD; ++m) a += (double)wc[m] * (double)feat[m * WD + k];
        put(d, WD, n, k, (float)a);
      }
      double bb = (double)bc[n];
      for (int m = 0; m < WD; ++m) bb += (double)wc[m] * (double)feat[WD * WD + m];
      put_hi_lo(d, WD, n, WD, (float)bb);
      for (int i = 0; i < kPeD; ++i) put(d, WD, n, WD + 2 + i, wc[WD + i]);
    }
  }
  {
    // both heads are ONE operand with K = 2 WD against A = [h | colour activation]: row 3 = density (reads h),
    // rows 0-2 = rgb (read the colour activation); L.dens is the second half of the same block
    uint16_t* d = (uint16_t*)(dst + L.rgb);
    for (int k = 0; k < WD; ++k) put(d, S::NHEAD, 3, k, dens[k]);
    for (int n = 0; n < 3; ++n)
      for (int k = 0; k < WD; ++k) put(d, S::NHEAD, n, WD + k, rgb[n * WD + k]);
    float hb[4] = {rgb[3 * WD + 0], rgb[3 * WD + 1], rgb[3 * WD + 2], dens[WD]};
    std::memcpy(dst + L.head_bias, hb, sizeof(hb));
  }
}

}  // namespace

size_t tc_pack_stride(const NetShape& net) {
  if (net.Lp != kLp || net.Ld != kLd) return 0;      // tensor path: paper's PE sizes only
  if (net.Wd == 32) return (size_t)make_tc_layout<32>(net.Hd).total;
  if (net.Wd == 64) return (size_t)make_tc_layout<64>(net.Hd).total;
  return 0;
}

// operand_f16: 0 = bfloat16 operands, 1 = binary16 operands.  Returns false if a value does not fit binary16.
bool tc_pack_subfield(const NetShape& net, const float* src_blob, void* dst, int operand_f16) {
  PackFmt fmt{operand_f16, false};
  if (net.Wd == 32) pack_subfield_t<32>(net, src_blob, dst, fmt);
  else if (net.Wd == 64) pack_subfield_t<64>(net, src_blob, dst, fmt);
  return !fmt.overflow;
}

// ---------------------------------------------------------------------------------------------
using namespace tc;

// heads of the bf16 path: ex2/lg2/rcp approximations (relative error ~2^-22, far below bf16)
// exp2 / log2 with denormals flushed: __expf / __logf guard the denormal range with a compare and two predicated
// multiplies each, and 1 + (a value below 2^-126) is 1 either way, so the results are the same bits
__device__ __forceinline__ float ex2_ftz(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float fast_sigmoid(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + ex2_ftz(x * -1.4426950408889634f)));
  return r;
}
__device__ __forceinline__ float fast_softplus(float x) {
  float l;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l) : "f"(1.0f + ex2_ftz(x * 1.4426950408889634f)));
  return x > 20.0f ? x : l * 0.6931471805599453f;        // a select, not a branch
}

// trunk-1 A row: [F(q) (63), 1] as 32 bf16x2 words, generated level by level with the double-angle
// recurrence and stored K step by K step (16 values = 8 TMEM columns), so that few values are live.
template <bool F16>
__device__ __forceinline__ void store_pe_row(uint32_t tA, const float q[3]) {
  // The row holds sin and TWICE the cosine of every level (the host halves the matching weight columns, which is
  // exact in bf16), because the double-angle step on (s, g = 2c) is s' = g s, g' = g g - 2: two operations per
  // level.  x and y advance together in packed binary32 pairs (add/mul/fma.f32x2: one issue slot for two lanes of
  // the FMA pipe, which this kernel leaves three quarters idle while it is short of issue slots); z is the pair
  // (s, g) with (s', g') = g (s, g) + (0, -2): one operation per level.
  float s[3], c[3];                               // c = 2 cos
  uint64_t S2, G2;
  sin_2cos_unit2(pack_f32x2(q[0], q[1]), S2, G2);
  unpack_f32x2(S2, s[0], s[1]);
  unpack_f32x2(G2, c[0], c[1]);
  sin_2cos_unit(q[2], s[2], c[2]);
  const uint64_t M2 = pack_f32x2(-2.0f, -2.0f), M02 = pack_f32x2(0.0f, -2.0f);
  float buf[16];
#pragma unroll
  for (int idx = 0; idx < 64; ++idx) {
    float v;
    if (idx < 3) {
      v = q[idx];
    } else if (idx == 63) {
      v = 1.0f;                                   // meets the bias row of B
    } else {
      const int l = (idx - 3) / 6, r = (idx - 3) % 6;
      if (r == 0 && l > 0) {                      // next level
        S2 = mul_f32x2(G2, S2);
        G2 = fma_f32x2(G2, G2, M2);
        unpack_f32x2(S2, s[0], s[1]);
        unpack_f32x2(G2, c[0], c[1]);
        unpack_f32x2(fma_f32x2(pack_f32x2(c[2], c[2]), pack_f32x2(s[2], c[2]), M02), s[2], c[2]);
      }
      v = r < 3 ? s[r] : c[r - 3];
    }
    buf[idx & 15] = v;
    if ((idx & 15) == 15) {
      uint32_t a8[8];
#pragma unroll
      for (int p = 0; p < 8; ++p) a8[p] = pack16<F16>(buf[2 * p], buf[2 * p + 1]);
      tmem_st_x8(tA + 8 * (idx >> 4), a8);
    }
  }
}

template <int WD, bool F16>
__global__ void __launch_bounds__(TcShape<WD>::kGroups * kTileRows, 1)
k_mlp_tc(GridParams g, FrameParams f, ChunkBuffers b, NetShape net, TcLayout lay,
         const unsigned char* __restrict__ wpack, const SubfieldFrame* __restrict__ frames, int n_bins,
         int spt) {
  using S = TcShape<WD>;
  constexpr int G = S::kGroups;
  extern __shared__ __align__(128) unsigned char smem_all[];   // G weight buffers of lay.total bytes
  __shared__ __align__(8) uint64_t bar_w_s[G], bar_d_s[G];
  __shared__ uint32_t tmem_base_s;
  // the NEXT tile's segment records, copied asynchronously while this tile runs (two buffers per group)
  constexpr int kStageSegs = 32;                               // staging serves K >= 4 (at most 32 segments per tile)
  __shared__ __align__(16) uint4 rec_stage_s[G][2][kStageSegs * kRecWords];
  // group and warp index are the same in every lane of a warp: broadcast from lane 0 so that everything derived
  // from them (TMEM columns, weight buffer, barriers, tile range) can live in uniform registers (measured: 5 %)
  const int grp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 7), 0);
  const int tid = threadIdx.x & (kTileRows - 1);
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  if (chunk_cancelled(b)) return;                              // (before anything is allocated)
  const unsigned total_tiles = (unsigned)b.totals[kTotTiles];
  const unsigned n_groups = gridDim.x * G;
  const unsigned per = (total_tiles + n_groups - 1) / n_groups;
  if ((unsigned)blockIdx.x * G * per >= total_tiles) return;   // whole CTA idle: nothing allocated yet
  const unsigned tile0 = min(total_tiles, (blockIdx.x * G + grp) * per);
  const unsigned tile1 = min(total_tiles, tile0 + per);

  uint64_t* const bar_w = &bar_w_s[grp];
  uint64_t* const bar_d = &bar_d_s[grp];
  unsigned char* const sw = smem_all + (size_t)grp * lay.total;
  if (tid == 0) {
    mbar_init(bar_w, 1);
    mbar_init(bar_d, 1);
    mbar_fence_init();
  }
  if (threadIdx.x < 32) tmem_alloc<512>(&tmem_base_s);
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tbase = __shfl_sync(0xffffffffu, tmem_base_s, 0);
  const uint32_t colG = (uint32_t)grp * S::G_COLS;               // this group's columns
  // warp w touches lanes 32w..32w+31.  The address is the same in every lane of a warp; broadcasting it from
  // lane 0 lets ptxas keep it in a uniform register (tcgen05.ld/st take their address from one): 3 % faster
  const uint32_t tA = __shfl_sync(0xffffffffu, tbase + ((uint32_t)(warp * 32) << 16) + colG, 0);
  const uint32_t tD = tA + S::D0;
  const uint32_t mA = tbase + colG, mD = mA + S::D0;           // MMA operand addresses (lane 0)

  const uint32_t sw_addr = smem_u32(sw);
  const uint32_t idesc_w = instr_desc_16(128, WD, F16), idesc_h = instr_desc_16(128, S::NHEAD, F16);
  const uint32_t bar_id = (uint32_t)grp + 1;
  // warp w of every group runs on scheduler w.  The warp that issues the MMAs and the one that stages the next
  // tile's records carry extra instructions, so both roles rotate with the group: each scheduler then hosts the
  // same number of issuing and staging warps instead of scheduler 0 all issuers and scheduler 3 all stagers
  const int iss_warp = grp & 3, stg_warp = (grp + 2) & 3;
  uint32_t par_d = 0, par_w = 0;
  const int K = g.K;
  const int sidx = tid / K, j = tid - sidx * K;
  float jf = (float)j + 0.5f;
  asm volatile("" : "+f"(jf));              // kept in its register: ptxas otherwise rebuilds it from the thread index in every tile

  // MMAs of one operand pair: ks K steps, A from TMEM columns a_col.., B blocks of N rows at b_off
  // The group's weight buffer never moves, so a block's descriptor is the buffer's plus the block's offset in
  // 16-byte units -- and every offset is a compile-time constant up to the number of trunk layers: two base values
  // (the buffer, the colour block) live in uniform registers and nothing is loaded or shifted between the group
  // barrier and the first tcgen05.mma of a layer (that stretch is on the critical path of every layer).
  constexpr uint32_t kT1 = (S::KP1 / 16) * S::blk(WD) / 16, kTS = (S::KH / 16) * S::blk(WD) / 16;   // trunk[1], stride
  constexpr uint32_t kRgb = (S::KC / 16) * S::blk(WD) / 16;                                         // heads
  const uint64_t desc0 = smem_desc(sw_addr, 128, 256);
  const uint32_t desc_hi = (uint32_t)(desc0 >> 32);
  const uint32_t dl0 = (uint32_t)desc0, dlc = dl0 + kT1 + (uint32_t)(net.Hd - 1) * kTS;
  auto mma_steps = [&](uint32_t d_col, uint32_t a_col, uint32_t lo, int N, uint32_t idesc, auto ks_c) {
    constexpr int ks = decltype(ks_c)::value;
#pragma unroll
    for (int s = 0; s < ks; ++s)
      mma_ts(d_col, a_col + 8 * s, ((uint64_t)desc_hi << 32) | (lo + (uint32_t)(s * (S::blk(N) >> 4))), idesc, s > 0);
  };
  // publish this thread's A row to the group's issuing thread
  auto publish = [&]() {
    wait_st();
    fence_before_sync();
    group_sync_r(bar_id);
  };
  auto wait_acc = [&]() {
    asm volatile("" : "+r"(par_d));          // in a vector register: nothing is moved inside the spin loop
    mbar_wait(bar_d, par_d);
    par_d ^= 1;
    fence_after_sync();
  };
  // D[0..WD) -> ReLU -> bf16x2 -> WD/2 columns at dst
  auto d_to_a = [&](uint32_t dst) {
#pragma unroll
    for (int h = 0; h < WD; h += 32) {
      uint32_t d[32];
      tmem_ld_x32(tD + h, d);
      wait_ld();
      uint32_t a[16];
#pragma unroll
      for (int c = 0; c < 16; ++c) a[c] = pack16_relu<F16>(__uint_as_float(d[2 * c]), __uint_as_float(d[2 * c + 1]));
      tmem_st_x16(dst + h / 2, a);
    }
  };

  unsigned k_tile_end = 0, k_tile_begin = 0, k_seg_begin = 0, k_seg_end = 0;
  bool have_k = false, staged = false;
  int stage_buf = 0;
  SubfieldFrame fr = frames[0];
  for (unsigned tile = tile0; tile < tile1; ++tile) {
    if (tile >= k_tile_end || !have_k) {
      // subfield of this tile: last k with tile_start[k] <= tile (a group's tiles are contiguous, so
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
      // stage the subfield's weights (TMA bulk copy); every MMA that read the old ones has completed,
      // because each thread has waited on the last layer's commit
      group_sync_r(bar_id);
      if (tid == 0) {
        mbar_expect_tx(bar_w, (uint32_t)lay.total);
        bulk_g2s(sw, wpack + (size_t)k * lay.total, (uint32_t)lay.total, bar_w);
      }
      have_k = true;
      mbar_wait(bar_w, par_w);
      par_w ^= 1;
    }
    const unsigned seg0 = k_seg_begin + (tile - k_tile_begin) * spt;
    const unsigned nseg = min((unsigned)spt, k_seg_end - seg0);
    const bool active = (unsigned)sidx < nseg;
    SegRec rec = make_uint4(0, 0, 0, 0);
    uint4 rd = make_uint4(0, 0, 0, 0);
    if (active) {
      if (staged) {                                          // copied to shared memory during the previous tile
        const uint4* sp = &rec_stage_s[grp][stage_buf][sidx * kRecWords];
        rec = sp[0];
        rd = sp[1];
      } else {
        const SegRec* rp = b.recs + (size_t)(seg0 + sidx) * kRecWords;
        rec = __ldg(rp);
        rd = __ldg(rp + 1);                                  // direction, pose
      }
    }
    // hide DRAM latency without registers: the next tile's records (same subfield, so their place is known) travel to shared memory with
    // cp.async and the records of the tile after it go to L2
    const bool stage_next = spt <= kStageSegs && tile + 1 < tile1 && tile + 1 < k_tile_end;
    // one warp (not the one that issues the MMAs) stages the next tile's records for the whole group: thread i of the
    // staging warp takes segment i (K >= 4: at most 32 segments per tile); the other three warps skip the block
    auto stage_records = [&]() {
      const int si = spt <= 32 ? tid - 32 * stg_warp : (j == 0 ? sidx : -1);
      if (si >= 0 && si < spt) {
        const unsigned sn = seg0 + spt + si;
        if (sn < k_seg_end) {
          if (stage_next) {
            uint4* dp = &rec_stage_s[grp][stage_buf ^ 1][si * kRecWords];
            cp_async_16(dp, b.recs + (size_t)sn * kRecWords);
            cp_async_16(dp + 1, b.recs + (size_t)sn * kRecWords + 1);
          }
          if (sn + spt < k_seg_end) prefetch_l2(b.recs + (size_t)(sn + spt) * kRecWords);
        }
      }
      cp_async_commit();
    };
    // width 32: behind the first layer's barrier (in front of it the staging warp reached the barrier last and the
    // whole group waited for it: 1.244 -> 1.214 ms on config 3); width 64, where the tensor pipe is the bound and a
    // group's four warps have a scheduler slot each to themselves: in front (behind it, config 4 was 4 % slower)
    constexpr bool kStageLate = WD == 32;
    if (!kStageLate) stage_records();
    const float* P = f.poses + rd.w * 12;
    const float t = __fmaf_rn(jf, __uint_as_float(rec.z), __uint_as_float(rec.y));   // reading D
    float q[3];                                              // reading A3
    q[0] = __fmul_rn(__fsub_rn(__fmaf_rn(t, __uint_as_float(rd.x), __ldg(P + 3)), fr.cx), fr.ix);
    q[1] = __fmul_rn(__fsub_rn(__fmaf_rn(t, __uint_as_float(rd.y), __ldg(P + 7)), fr.cy), fr.iy);
    q[2] = __fmul_rn(__fsub_rn(__fmaf_rn(t, __uint_as_float(rd.z), __ldg(P + 11)), fr.cz), fr.iz);
    if (!active) q[0] = q[1] = q[2] = 0.0f;                  // idle rows stay finite

    // ---- trunk-1: A = [F(q), 1]
    store_pe_row<F16>(tA, q);
    // the ray's direction block [1, 1, F(d), 0 0 0]: requested before the group barrier so that the load runs
    // behind the barrier, the MMA issue and the MMA itself (asked for after the issue it arrived later than the
    // accumulators: 4 % of the kernel's stall samples sat on the tcgen05.st below)
    uint32_t ad[16];
    {
      const uint4* db = b.dirblk + (size_t)rec.x * 4;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint4 v;
        asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(db + c));
        ad[4 * c] = v.x; ad[4 * c + 1] = v.y; ad[4 * c + 2] = v.z; ad[4 * c + 3] = v.w;
      }
    }
    publish();
    if (warp == iss_warp) {
      if (elect_one()) {
        fence_after_sync();
        mma_steps(mD, mA, dl0, WD, idesc_w, std::integral_constant<int, S::KP1 / 16>{});
        mma_commit(bar_d);
      }
      __syncwarp();
    }
    if (kStageLate) stage_records();
    wait_acc();
    tmem_st_x16(tA + S::A_FD, ad);                           // parks behind h for every later layer
    // ---- trunk-2..Hd: A = [h, 1, 1, ...]
    // (the loop runs on the descriptor itself: its end value is already in a uniform register, a comparison with
    // net.Hd would put a parameter load between the accumulator wait and the tcgen05.ld of the next layer)
#pragma unroll 1
    for (uint32_t dlt = dl0 + kT1; dlt != dlc; dlt += kTS) {
      d_to_a(tA + S::A_H);
      publish();
      if (warp == iss_warp) {
        if (elect_one()) {
          fence_after_sync();
          mma_steps(mD, mA, dlt, WD, idesc_w, std::integral_constant<int, S::KH / 16>{});
          mma_commit(bar_d);
        }
        __syncwarp();
      }
      wait_acc();
    }
    // ---- colour (feature layer folded in): A = [h, 1, 1, F(d), 0 0 0]
    d_to_a(tA + S::A_H);
    publish();
    if (warp == iss_warp) {
      if (elect_one()) {
        fence_after_sync();
        mma_steps(mD, mA, dlc, WD, idesc_w, std::integral_constant<int, S::KC / 16>{});
        mma_commit(bar_d);
      }
      __syncwarp();
    }
    wait_acc();
    // ---- heads: one N = 16 operand over A = [h | colour activation] (the activation takes the direction block's
    //      columns, h is still in place): outputs r, g, b, sigma in four adjacent accumulator columns
    d_to_a(tA + S::A_FD);
    cp_async_wait_all();                                     // the staged records are complete before this barrier
    publish();
    staged = stage_next;
    stage_buf ^= 1;
    if (warp == iss_warp) {
      if (elect_one()) {
        fence_after_sync();
        mma_steps(mD, mA + S::A_H, dlc + kRgb, S::NHEAD, idesc_h, std::integral_constant<int, 2 * WD / 16>{});
        mma_commit(bar_d);
      }
      __syncwarp();
    }
    const float4 hb = *reinterpret_cast<const float4*>(sw + lay.head_bias);
    wait_acc();
    uint32_t craw[4];                                        // r, g, b, sigma
    tmem_ld_x4(tD, craw);
    wait_ld();
    // ---- activations (A4), fp32
    const float sigma_raw = __uint_as_float(craw[3]) + hb.w;
    // a sample leaves as four binary16 values (sigma clamped to the largest finite one): 8 bytes
    const float sigma = fminf(net.act == 1 ? fast_softplus(sigma_raw) : fmaxf(sigma_raw, 0.0f), 65504.0f);
    uint2 o2;
    o2.x = pack_f16(sigma, fast_sigmoid(__uint_as_float(craw[0]) + hb.x));
    o2.y = pack_f16(fast_sigmoid(__uint_as_float(craw[1]) + hb.y), fast_sigmoid(__uint_as_float(craw[2]) + hb.z));
    if (active) reinterpret_cast<uint2*>(b.out)[(size_t)rec.w * K + __float2int_rz(jf)] = o2;
  }
  fence_before_sync();
  __syncthreads();
  if (threadIdx.x < 32) tmem_dealloc<512>(tbase);
}

template <int WD, bool F16>
static cudaError_t launch_tc_t(const GridParams& g, const FrameParams& f, const ChunkBuffers& b,
                               const NetShape& net, const void* wpack, const SubfieldFrame* frames, int n_bins,
                               int spt, int n_sms, cudaStream_t s) {
  using S = TcShape<WD>;
  if (!b.dirblk) return cudaErrorInvalidValue;
  TcLayout lay = make_tc_layout<WD>(net.Hd);
  // one CTA per SM owns all 512 TMEM columns; asking for more than half of the shared memory keeps a
  // second CTA (which would block in tcgen05.alloc) off the SM
  size_t smem = (size_t)S::kGroups * lay.total;
  if (smem < 120 * 1024) smem = 120 * 1024;
  if (smem > 227 * 1024) return cudaErrorInvalidValue;
  cudaError_t e = cudaFuncSetAttribute(k_mlp_tc<WD, F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_mlp_tc<WD, F16><<<n_sms, S::kGroups * kTileRows, smem, s>>>(g, f, b, net, lay, (const unsigned char*)wpack, frames,
                                                               n_bins, spt);
  return cudaGetLastError();
}

cudaError_t launch_mlp_tc(const GridParams& g, const FrameParams& f, const ChunkBuffers& b, const NetShape& net,
                          const void* wpack, size_t wpack_stride, int operand_f16, const SubfieldFrame* frames,
                          int n_bins, int segs_per_tile, int n_sms, cudaStream_t s) {
  if (!wpack || wpack_stride == 0) return cudaErrorNotSupported;
  if (net.Wd == 32 && !operand_f16) return launch_tc_t<32, false>(g, f, b, net, wpack, frames, n_bins, segs_per_tile, n_sms, s);
  if (net.Wd == 32) return launch_tc_t<32, true>(g, f, b, net, wpack, frames, n_bins, segs_per_tile, n_sms, s);
  if (net.Wd == 64 && !operand_f16) return launch_tc_t<64, false>(g, f, b, net, wpack, frames, n_bins, segs_per_tile, n_sms, s);
  if (net.Wd == 64) return launch_tc_t<64, true>(g, f, b, net, wpack, frames, n_bins, segs_per_tile, n_sms, s);
  return cudaErrorInvalidValue;
}

// dynamic + static shared memory the tensor kernel needs for this network; 0 if the tensor path does not apply
size_t tc_smem_bytes(const NetShape& net) {
  if (net.Lp != kLp || net.Ld != kLd) return 0;
  if (net.Wd == 32) return (size_t)TcShape<32>::kGroups * make_tc_layout<32>(net.Hd).total + 20 * 1024;
  if (net.Wd == 64) return (size_t)TcShape<64>::kGroups * make_tc_layout<64>(net.Hd).total + 12 * 1024;
  return 0;
}

}  // namespace r360
