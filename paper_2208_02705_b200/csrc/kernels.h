// r360 -- host-side launch wrappers of the CUDA kernels (one per pipeline stage).
#pragma once
#include "common.cuh"
#include "pe.cuh"

namespace r360 {

// Per-subfield constants in device memory.
struct SubfieldFrame {      // reading A3: q = (p - centre) * inv_half
  float cx, cy, cz, pad0;
  float ix, iy, iz, pad1;
};

// Network shape shared by the MLP kernels.
struct NetShape {
  int Wd;        // hidden width (32 / 64)
  int Hd;        // trunk layers
  int Lp, Ld;    // PE levels
  int pe_p, pe_d;
  int act;       // 0 ReLU, 1 softplus
  int P;         // parameters per subfield (fp32 blob, transposed layout has the same size)
};

// Device layout of one subfield's fp32 weights for the ALU kernel (float offsets; every block
// is padded to a multiple of 4 floats so rows can be read as float4):
//   trunk l : W^T[in][Wd] then b[Wd]        density : w[Wd] then b, pad 3
//   feature : W^T[Wd][Wd] then b[Wd]        colour  : W^T[Wd+pe_d][Wd] then b[Wd]
//   rgb     : W^T[Wd][4] (r,g,b,0) then b[4]
struct Fp32Layout {
  int trunk[8];
  int dens, feat, col, rgb;
  int total;
};

// Device buffers of one ray chunk.
struct ChunkBuffers {
  uint32_t* ray_cnt;     // [n_rays] segments per ray
  uint32_t* ray_off;     // [n_rays] block-local exclusive offset after count; global after emit
  uint32_t* block_sum;   // [n_blocks] segments per sampler block -> exclusive scan in place
  uint32_t* bin_cnt;     // [n] segments per subfield reserved by sampler blocks (k_count); total after k_scan
  uint32_t* bin_ovf;     // [n] segments per subfield that no block reserved (a block's list was full)
  uint2* blk_list;       // [n_blocks][kBlkListCap] (subfield, first position inside its bin) reserved by the block
  uint32_t* blk_list_n;  // [n_blocks] entries used
  uint32_t* bin_start;   // [n+1]
  uint32_t* bin_cursor;  // [n]
  uint32_t* tile_start;  // [n+1] first MLP tile of each subfield
  unsigned long long* totals;  // [kTotN] device-side counters of the current ray chunk (indices below)
  unsigned long long* host_flags;  // mapped pinned host memory, [2]: k_scan posts {overflow flag, largest pass} of the
                                   // chunk here, so the host learns them without a copy in the stream
  float2* seg_td;        // [G] ray-major (t_in, delta) of every segment: one 8-byte access per segment and lane
  SegRec* recs;          // [G * kRecWords] binned by subfield (common.cuh: SegRec)
  float4* out;           // [G*K] (sigma, r, g, b) per sample, ray-major; the tensor path stores a sample as four
                         // binary16 values (8 bytes, the same buffer read as uint2)
  // first kHitCap hits of every ray, kept by k_count so that k_emit re-walks only the rays with more
  float2* hit_t;         // [kHitCap][n_rays] (t_in, delta)
  uint16_t* hit_lab;     // [kHitCap][n_rays]
  // wavefront passes only (r360_set_wavefront; null otherwise):
  uint32_t* pass_cnt;    // [n_rays] segments of the ray in the current pass
  uint32_t* pass_off;    // [n_rays] first ray-major slot of the ray in the current pass
  float4* st_c;          // [n_rays] compositing state carried between passes: C_r, C_g, C_b, D
  float* st_T;           // [n_rays] transmittance carried between passes; < 0 = the ray is finished
  // tensor path only (null otherwise):
  uint4* dirblk;         // [n_rays*4] per ray: [1, 1, F(d), 0..] as 32 values in the operand format (pe.cuh)
  int dir_f16;           // operand format of dirblk: 0 bfloat16, 1 binary16
};

// ChunkBuffers::totals, reset at the start of every ray chunk.  The kernels that follow k_scan size nothing on
// the host: they read the counts from here, and they return at once when kTotOverflow is set (the chunk's
// segments exceed the capacity of the segment buffers: the host re-renders the chunk with larger buffers, see
// render.cu) or when kTotWaveDone is set (wavefront: every ray has finished, the remaining passes have no work).
enum : int {
  kTotSegs = 0,       // segments of the current pass (k_scan)
  kTotTiles = 1,      // MLP tiles of the current pass (k_scan)
  kTotUsed = 2,       // samples composited before early-out, summed over the chunk's passes (k_composite)
  kTotGeo = 3,        // wavefront: occupied voxels crossed by all rays (k_count); single pass: unused
  kTotOverflow = 4,   // sticky: a pass had more segments than seg_cap
  kTotWaveDone = 5,   // sticky: a wavefront pass after the first had no segments
  kTotSegSum = 6,     // segments summed over the chunk's passes
  kTotTileSum = 7,    // tiles summed over the chunk's passes
  kTotSegMax = 8,     // largest pass of the chunk, in segments (sizes the buffers of later frames)
  kTotN = 16
};
__device__ __forceinline__ bool chunk_cancelled(const ChunkBuffers& b) {
  return (b.totals[kTotOverflow] | b.totals[kTotWaveDone]) != 0;
}

#ifndef R360_SAMPLER_THREADS
#define R360_SAMPLER_THREADS 256
#endif
constexpr int kSamplerThreads = R360_SAMPLER_THREADS;   // rays per sampler block (k_count, k_emit, k_pass_count)

// Wavefronted early termination: the hits of a ray are fed to the MLP in passes
// [h0, h1) = [0,2) [2,6) [6,16) [16,kHitCap) [kHitCap, inf); after every pass the compositing kernel retires
// the rays whose transmittance fell below tau, so their remaining samples never reach the MLP.  The passes
// inside the hit buffer replay it; the tail pass walks again (only rays still alive with more hits than the
// buffer holds).  All zero in the single-pass path.
struct PassParams {
  int wavefront;
  int first, last;
  uint32_t h0, h1;
};
constexpr int kHitCap = 64;
constexpr int kBlkListCap = 256;

void launch_count(const GridParams& g, const uint16_t* grid, const FrameParams& f, const ChunkBuffers& b,
                  int n_bins, cudaStream_t s);
// seg_cap: capacity of the segment buffers (seg_td, recs, out) in segments; later_wave_pass: a wavefront
// pass after the first (an empty one ends the chunk)
void launch_scan(const ChunkBuffers& b, int n_blocks, int n_bins, int segs_per_tile, unsigned long long seg_cap,
                 int later_wave_pass, cudaStream_t s);
void launch_emit(const GridParams& g, const uint16_t* grid, const FrameParams& f, const ChunkBuffers& b,
                 int n_bins, const PassParams& pp, cudaStream_t s);
// wavefront: segments of every ray in this pass, block-local offsets, the pass's histogram and reservations
void launch_pass_count(const GridParams& g, const uint16_t* grid, const FrameParams& f, const ChunkBuffers& b,
                       int n_bins, const PassParams& pp, cudaStream_t s);
// fp32 MLP on the FP32 ALUs.  weights_t: per subfield, per layer W^T[in][out] then b[out].
cudaError_t launch_mlp_fp32(const GridParams& g, const FrameParams& f, const ChunkBuffers& b,
                            const NetShape& net, const Fp32Layout& lay, const float* weights_t,
                            const SubfieldFrame* frames, int n_bins, int segs_per_tile, int n_sms,
                            cudaStream_t s);
// 16-bit tensor-core MLP (tcgen05, fp32 accumulate).  wpack: per subfield packed operand tiles (bfloat16, or
// binary16 when operand_f16) + fp32 head biases.
cudaError_t launch_mlp_tc(const GridParams& g, const FrameParams& f, const ChunkBuffers& b,
                          const NetShape& net, const void* wpack, size_t wpack_stride, int operand_f16,
                          const SubfieldFrame* frames, int n_bins, int segs_per_tile, int n_sms,
                          cudaStream_t s);
void launch_composite(const GridParams& g, const FrameParams& f, const ChunkBuffers& b, float tau,
                      void* out_rgb, void* out_depth, const PassParams& pp, bool half_samples, cudaStream_t s);
// debug: expand binned records into ray-major per-sample t and subfield id
void launch_export_samples(const GridParams& g, const ChunkBuffers& b, int n_bins, unsigned n_segs,
                           float* t, int32_t* subfield, cudaStream_t s);
void launch_export_field(const ChunkBuffers& b, size_t n_samples, bool half_samples, float* field, cudaStream_t s);
void launch_export_counts(const ChunkBuffers& b, unsigned n_rays, int K, uint32_t* counts, uint32_t* offsets,
                          cudaStream_t s);

}  // namespace r360
