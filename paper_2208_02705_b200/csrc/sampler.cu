// r360 -- ray generation + occupancy walk sampler, and the binning by subfield (steps a1-a5).
//
//   k_count : one walk per ray (exact empty-space skipping, common.cuh: Walker) -> segments per ray, block-local
//             exclusive offsets, the first kHitCap hits of every ray in a ray-major hit buffer, the ray's direction
//             block for the tensor path, the per-subfield histogram of the block and -- from it -- the block's
//             RESERVATION of a range in every bin it touched (one returning atomic per block and subfield)
//   k_scan  : one launch, two blocks: exclusive scan of the block sums; exclusive scan of the histogram (bin
//             starts) and of the per-subfield MLP tile counts
//   k_emit  : every segment goes to its bin: hits are replayed from the hit buffer and placed with shared-memory
//             cursors inside the block's reservations (no global atomics); only rays with more than kHitCap hits
//             walk again.  The ray-major (t_in, delta) pair is kept for the compositing kernel.
//   k_pass_count : the histogram / reservation step of one wavefront pass (r360_set_wavefront), from the hit buffer
// A "segment" is one occupied voxel crossed by one ray; it stands for K samples (reading D).
// PAPER.md:174 (ray casting to localise occupied voxels, per-voxel tiny-MLP label), :164, :29.
#include "kernels.h"

namespace r360 {

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// Block-wide exclusive scan of one value per thread (blockDim.x = kSamplerThreads).
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t x, uint32_t* warp_sums, uint32_t& total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = x;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += y;
  }
  if (lane == 31) warp_sums[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = lane < (int)(blockDim.x >> 5) ? warp_sums[lane] : 0;
    uint32_t wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += y;
    }
    warp_sums[lane] = wi - w;          // exclusive warp offsets
    if (lane == 31) warp_sums[32] = wi;  // block total
  }
  __syncthreads();
  total = warp_sums[32];
  return warp_sums[wid] + incl - x;
}

// The block's bin reservations (made by k_count, or by k_pass_count for a wavefront pass) as shared-memory
// cursors: cur[k] = next position of this block inside bin k, kNotReserved if the block reserved nothing.
constexpr uint32_t kNotReserved = 0xFFFFFFFFu;

__device__ __forceinline__ void load_reservations(const ChunkBuffers& b, uint32_t* cur, int n_bins) {
  for (int k = threadIdx.x; k < n_bins; k += blockDim.x) cur[k] = kNotReserved;
  __syncthreads();
  const uint2* list = b.blk_list + (size_t)blockIdx.x * kBlkListCap;
  const uint32_t n = b.blk_list_n[blockIdx.x];
  for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
    const uint2 e = list[i];
    cur[e.x] = __ldg(b.bin_start + e.x) + e.y;
  }
  __syncthreads();
}

// The block's histogram -> one returning atomic per subfield present, remembered in the block's list.
__device__ __forceinline__ void reserve_bins(const ChunkBuffers& b, const uint32_t* hist, int n_bins) {
  __shared__ uint32_t list_n;
  if (threadIdx.x == 0) list_n = 0;
  __syncthreads();
  uint2* list = b.blk_list + (size_t)blockIdx.x * kBlkListCap;
  for (int k = threadIdx.x; k < n_bins; k += blockDim.x) {
    const uint32_t c = hist[k];
    if (c) {
      const uint32_t i = atomicAdd(&list_n, 1u);
      if (i < (uint32_t)kBlkListCap) list[i] = make_uint2((uint32_t)k, atomicAdd(&b.bin_cnt[k], c));
      else atomicAdd(&b.bin_ovf[k], c);          // list full: k_emit falls back to the global cursor
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) b.blk_list_n[blockIdx.x] = min(list_n, (uint32_t)kBlkListCap);
}

// ---------------------------------------------------------------------------------------
// DIR: 0 = no direction blocks (fp32 path), 1 = bfloat16, 2 = binary16 (a template parameter: with a run-time
// format the two conversion paths cost the walk six registers and a resident block per SM)
template <int DIR>
__global__ void __launch_bounds__(kSamplerThreads)
k_count(GridParams g, const uint16_t* __restrict__ grid, FrameParams f, ChunkBuffers b, int n_bins,
        int use_smem_hist) {
  extern __shared__ uint32_t hist[];     // [n_bins] when use_smem_hist
  __shared__ uint32_t warp_sums[33];
  if (use_smem_hist) {
    for (int k = threadIdx.x; k < n_bins; k += blockDim.x) hist[k] = 0;
    __syncthreads();
  }
  const unsigned r = blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = r < f.n_rays;
  Walker w;
  w.alive = false;
  if (valid) {
    const Ray ray = make_ray(f, r);
    w.init(g, ray);
    if constexpr (DIR != 0) store_dir_block<DIR == 2>(b.dirblk + (size_t)r * 4, ray.d);   // tensor path: F(d) once per ray
  }
  uint32_t cnt = 0;
  // lock-step over "next occupied voxel" so the histogram update can be warp-aggregated
  while (__any_sync(0xffffffffu, w.alive)) {
    uint32_t lab = 0;
    float t_in, t_out;
    // one walk iteration per lane and round: a lane that has found a voxel goes on with the others instead of
    // waiting for them to find theirs
    const bool hit = w.alive && w.advance(g, grid, lab, t_in, t_out);
    unsigned m = __ballot_sync(0xffffffffu, hit);
    if (m == 0) continue;
    if (hit) {
      if (cnt < kHitCap) {
        // reading D: delta = (t_out - t_in) / K, one subtract, one divide
        const size_t h = (size_t)cnt * f.n_rays + r;
        b.hit_t[h] = make_float2(t_in, seg_delta(g, t_in, t_out));
        b.hit_lab[h] = (uint16_t)lab;
      }
      ++cnt;
      if (!b.pass_cnt) {      // (wavefront: every pass builds its own histogram, k_pass_count)
        unsigned peers = __match_any_sync(m, lab);
        if ((peers & lanemask_lt()) == 0) {
          uint32_t c = __popc(peers);
          if (use_smem_hist) atomicAdd(&hist[lab], c);
          else atomicAdd(&b.bin_ovf[lab], c);
        }
      }
    }
  }
  uint32_t total;
  uint32_t off = block_exclusive_scan(cnt, warp_sums, total);
  if (valid) {
    b.ray_cnt[r] = cnt;
    b.ray_off[r] = off;
  }
  if (threadIdx.x == 0) b.block_sum[blockIdx.x] = total;
  if (b.pass_cnt) {
    if (threadIdx.x == 0 && total) atomicAdd(&b.totals[kTotGeo], (unsigned long long)total);   // geometric segments
    return;
  }
  if (use_smem_hist) {
    // The block RESERVES its share of every bin it touched: one returning atomic per (block, subfield),
    // remembered in the block's list, so that k_emit places this block's segments with shared-memory
    // cursors and no global atomics (thousands of warps hit the same few subfields at the same time).
    __syncthreads();
    reserve_bins(b, hist, n_bins);
  } else if (threadIdx.x == 0) {
    b.blk_list_n[blockIdx.x] = 0;
  }
}

// ---------------------------------------------------------------------------------------
// Single-block exclusive scan over m values (in -> out, may alias); returns the total to all
// threads.  blockDim.x = 1024.
__device__ uint64_t scan_array(const uint32_t* in, uint32_t* out, int m, uint32_t* sm /*[34]*/,
                               int tile_div /*0: raw values; >0: scan ceil(v/tile_div)*/,
                               const uint32_t* src_for_tiles) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint64_t carry = 0;
  for (int base = 0; base < m; base += 1024) {
    int i = base + threadIdx.x;
    uint32_t x = 0;
    if (i < m) {
      x = tile_div ? (src_for_tiles[i] + tile_div - 1) / tile_div : in[i];
    }
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += y;
    }
    if (lane == 31) sm[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      uint32_t w = sm[lane], wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, wi, o);
        if (lane >= o) wi += y;
      }
      sm[lane] = wi - w;
      if (lane == 31) sm[32] = wi;
    }
    __syncthreads();
    if (i < m) out[i] = (uint32_t)(carry + sm[wid] + incl - x);
    carry += sm[32];
    __syncthreads();
  }
  return carry;
}

__global__ void __launch_bounds__(1024)
k_scan(ChunkBuffers b, int n_blocks, int n_bins, int segs_per_tile, unsigned long long seg_cap, int later_wave_pass) {
  __shared__ uint32_t sm[34];
  if (later_wave_pass && chunk_cancelled(b)) return;       // an earlier pass overflowed or ended the chunk
  if (blockIdx.x == 0) {
    uint64_t tot = scan_array(b.block_sum, b.block_sum, n_blocks, sm, 0, nullptr);
    if (threadIdx.x == 0) {
      // one thread, stream order: plain read-modify-writes
      b.totals[kTotSegs] = tot;
      b.totals[kTotSegSum] += tot;
      if (tot > b.totals[kTotSegMax]) b.totals[kTotSegMax] = tot;
      if (tot > seg_cap) b.totals[kTotOverflow] = 1;
      if (later_wave_pass && tot == 0) b.totals[kTotWaveDone] = 1;
      b.host_flags[0] = b.totals[kTotOverflow];
      b.host_flags[1] = b.totals[kTotSegMax];
      __threadfence_system();
    }
  } else {
    // a bin = [segments reserved by blocks | the rest, placed through the global cursor]
    for (int k = threadIdx.x; k < n_bins; k += blockDim.x) {
      const uint32_t res = b.bin_cnt[k];
      b.bin_cursor[k] = res;
      b.bin_cnt[k] = res + b.bin_ovf[k];
    }
    __syncthreads();
    // tile counts first (they read bin_cnt), then the bin starts
    uint64_t tiles = scan_array(nullptr, b.tile_start, n_bins, sm, segs_per_tile, b.bin_cnt);
    uint64_t segs = scan_array(b.bin_cnt, b.bin_start, n_bins, sm, 0, nullptr);
    if (threadIdx.x == 0) {
      b.tile_start[n_bins] = (uint32_t)tiles;
      b.bin_start[n_bins] = (uint32_t)segs;
      b.totals[kTotTiles] = tiles;
      b.totals[kTotTileSum] += tiles;
    }
  }
}

// ---------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------
// Wavefront pass: how many segments each ray contributes to this pass, block-local offsets, and the pass's
// histogram / reservations.  Passes inside the hit buffer read the labels from it; the tail pass (hits beyond
// the buffer, rays still alive only) walks again and skips the buffered hits.
__global__ void __launch_bounds__(kSamplerThreads)
k_pass_count(GridParams g, const uint16_t* __restrict__ grid, FrameParams f, ChunkBuffers b, int n_bins,
             int use_smem_hist, PassParams pp) {
  extern __shared__ uint32_t hist[];
  __shared__ uint32_t warp_sums[33];
  if (chunk_cancelled(b)) return;
  if (use_smem_hist) {
    for (int k = threadIdx.x; k < n_bins; k += blockDim.x) hist[k] = 0;
    __syncthreads();
  }
  const unsigned r = blockIdx.x * blockDim.x + threadIdx.x;
  const bool tail = pp.h0 >= (uint32_t)kHitCap;
  uint32_t m = 0;                      // segments of this ray in this pass
  if (r < f.n_rays) {
    const uint32_t cnt = b.ray_cnt[r];
    if ((pp.first || b.st_T[r] >= 0.0f) && cnt > pp.h0) m = min(cnt, pp.h1) - pp.h0;
    b.pass_cnt[r] = m;
  }
  uint32_t total;
  const uint32_t off = block_exclusive_scan(m, warp_sums, total);
  if (r < f.n_rays) b.ray_off[r] = off;
  if (threadIdx.x == 0) b.block_sum[blockIdx.x] = total;
  auto tally = [&](bool hit, uint32_t lab) {
    const unsigned msk = __ballot_sync(0xffffffffu, hit);
    if (hit) {
      const unsigned peers = __match_any_sync(msk, lab);
      if ((peers & lanemask_lt()) == 0) {
        const uint32_t c = __popc(peers);
        if (use_smem_hist) atomicAdd(&hist[lab], c);
        else atomicAdd(&b.bin_ovf[lab], c);
      }
    }
  };
  if (!tail) {
    uint32_t m_max = m;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m_max = max(m_max, __shfl_xor_sync(0xffffffffu, m_max, o));
    for (uint32_t h = 0; h < m_max; ++h) {
      const bool hit = h < m;
      tally(hit, hit ? (uint32_t)b.hit_lab[(size_t)(pp.h0 + h) * f.n_rays + r] : 0u);
    }
  } else {
    Walker w;
    w.alive = false;
    if (m) w.init(g, make_ray(f, r));
    uint32_t seen = 0;
    while (__any_sync(0xffffffffu, w.alive)) {
      uint32_t lab = 0;
      float t_in, t_out;
      bool hit = w.alive && w.advance(g, grid, lab, t_in, t_out);
      if (hit && seen++ < (uint32_t)kHitCap) hit = false;      // already processed from the hit buffer
      tally(hit, lab);
    }
  }
  if (use_smem_hist) {
    __syncthreads();
    reserve_bins(b, hist, n_bins);
  } else if (threadIdx.x == 0) {
    b.blk_list_n[blockIdx.x] = 0;
  }
}

// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kSamplerThreads)
k_emit(GridParams g, const uint16_t* __restrict__ grid, FrameParams f, ChunkBuffers b, int n_bins,
       int use_smem_cursor, PassParams pp) {
  extern __shared__ uint32_t cur[];      // [n_bins] when use_smem_cursor: next position of this block in each bin
  if (chunk_cancelled(b)) return;
  if (use_smem_cursor) load_reservations(b, cur, n_bins);
  const unsigned r = blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = r < f.n_rays;
  Walker w;
  w.alive = false;
  uint32_t slot = 0, cnt = 0, h = 0, h_end = 0, skip = 0;
  uint4 dir = make_uint4(0, 0, 0, 0);
  bool replay = true;
  if (valid) {
    const uint32_t cnt_total = b.ray_cnt[r];
    cnt = pp.wavefront ? b.pass_cnt[r] : cnt_total;      // segments of this ray in this launch
    slot = b.block_sum[blockIdx.x] + b.ray_off[r];
    if (pp.wavefront) b.pass_off[r] = slot;
    else b.ray_off[r] = slot;                              // now the global ray-major offset
    // single pass: replay if every hit of the ray is in the hit buffer, otherwise walk again; wavefront: the
    // passes inside the hit buffer replay, the tail pass walks and skips the buffered hits
    replay = pp.wavefront ? pp.h0 < (uint32_t)kHitCap : cnt_total <= (uint32_t)kHitCap;
    if (pp.wavefront && !replay) skip = kHitCap;
    if (cnt) {
      const Ray ray = make_ray(f, r);
      dir = make_uint4(__float_as_uint(ray.d[0]), __float_as_uint(ray.d[1]), __float_as_uint(ray.d[2]), ray.pose);
      if (replay) {
        h = pp.wavefront ? pp.h0 : 0u;
        h_end = h + cnt;
      } else {
        w.init(g, ray);                                    // otherwise walk again, all hits in one go
      }
    }
  }
  bool more = replay ? h < h_end : w.alive;
  // replay: the next hit is requested one round ahead, so two rounds of loads are in flight per lane
  float2 td_n = make_float2(0.f, 0.f);
  uint32_t lab_n = 0;
  if (replay && h < h_end) {
    const size_t i = (size_t)h * f.n_rays + r;
    td_n = b.hit_t[i];
    lab_n = b.hit_lab[i];
  }
  while (__any_sync(0xffffffffu, more)) {
    uint32_t lab = 0;
    float t_in = 0.f, dt = 0.f;
    bool hit = false;
    if (replay) {
      if (h < h_end) {
        t_in = td_n.x; dt = td_n.y;
        lab = lab_n;
        hit = true;
        ++h;
        if (h < h_end) {
          const size_t i = (size_t)h * f.n_rays + r;
          td_n = b.hit_t[i];
          lab_n = b.hit_lab[i];
        }
      }
      more = h < h_end;
    } else {
      float t_out = 0.f;
      hit = w.alive && w.advance(g, grid, lab, t_in, t_out);     // one walk iteration per round (see k_count)
      if (hit && skip) {                                   // tail pass: this hit was processed from the buffer
        --skip;
        hit = false;
      }
      if (hit) dt = seg_delta(g, t_in, t_out);    // reading D
      more = w.alive;
    }
    unsigned m = __ballot_sync(0xffffffffu, hit);
    if (hit) {
      unsigned peers = __match_any_sync(m, lab);
      int leader = __ffs(peers) - 1;
      uint32_t base = 0;
      if ((int)(threadIdx.x & 31) == leader) {
        const uint32_t c = (uint32_t)__popc(peers);
        if (use_smem_cursor && cur[lab] != kNotReserved) base = atomicAdd(&cur[lab], c);   // reserved by the block
        else base = __ldg(b.bin_start + lab) + atomicAdd(&b.bin_cursor[lab], c);
      }
      base = __shfl_sync(peers, base, leader);
      uint32_t pos = base + __popc(peers & lanemask_lt());
      b.recs[(size_t)pos * kRecWords] = make_uint4(r, __float_as_uint(t_in), __float_as_uint(dt), slot);
      b.recs[(size_t)pos * kRecWords + 1] = dir;
      b.seg_td[slot] = make_float2(t_in, dt);
      ++slot;
    }
  }
}

// ---------------------------------------------------------------------------------------
// debug taps
__global__ void k_export_samples(GridParams g, ChunkBuffers b, int n_bins, unsigned n_segs, float* t,
                                 int32_t* subfield) {
  unsigned pos = blockIdx.x * blockDim.x + threadIdx.x;
  if (pos >= n_segs) return;
  // subfield of a bin position: last k with bin_start[k] <= pos
  int lo = 0, hi = n_bins;
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (b.bin_start[mid] <= pos) lo = mid; else hi = mid;
  }
  SegRec rec = b.recs[(size_t)pos * kRecWords];
  float t_in = __uint_as_float(rec.y), dt = __uint_as_float(rec.z);
  size_t s0 = (size_t)rec.w * g.K;
  for (int j = 0; j < g.K; ++j) {
    t[s0 + j] = __fmaf_rn((float)j + 0.5f, dt, t_in);
    subfield[s0 + j] = lo;
  }
}

__global__ void k_export_counts(ChunkBuffers b, unsigned n_rays, int K, uint32_t* counts, uint32_t* offsets) {
  unsigned r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rays) return;
  counts[r] = b.ray_cnt[r] * K;
  offsets[r] = b.ray_off[r] * K;
}

// ---------------------------------------------------------------------------------------
void launch_count(const GridParams& g, const uint16_t* grid, const FrameParams& f, const ChunkBuffers& b,
                  int n_bins, cudaStream_t s) {
  int blocks = (f.n_rays + kSamplerThreads - 1) / kSamplerThreads;
  int use_smem = n_bins <= 8192;
  size_t smem = use_smem ? (size_t)n_bins * sizeof(uint32_t) : 0;
  if (!b.dirblk) k_count<0><<<blocks, kSamplerThreads, smem, s>>>(g, grid, f, b, n_bins, use_smem);
  else if (!b.dir_f16) k_count<1><<<blocks, kSamplerThreads, smem, s>>>(g, grid, f, b, n_bins, use_smem);
  else k_count<2><<<blocks, kSamplerThreads, smem, s>>>(g, grid, f, b, n_bins, use_smem);
}

void launch_scan(const ChunkBuffers& b, int n_blocks, int n_bins, int segs_per_tile, unsigned long long seg_cap,
                 int later_wave_pass, cudaStream_t s) {
  k_scan<<<2, 1024, 0, s>>>(b, n_blocks, n_bins, segs_per_tile, seg_cap, later_wave_pass);
}

void launch_emit(const GridParams& g, const uint16_t* grid, const FrameParams& f, const ChunkBuffers& b,
                 int n_bins, const PassParams& pp, cudaStream_t s) {
  int blocks = (f.n_rays + kSamplerThreads - 1) / kSamplerThreads;
  int use_smem = n_bins <= 8192;
  size_t smem = use_smem ? (size_t)n_bins * sizeof(uint32_t) : 0;
  k_emit<<<blocks, kSamplerThreads, smem, s>>>(g, grid, f, b, n_bins, use_smem, pp);
}

void launch_pass_count(const GridParams& g, const uint16_t* grid, const FrameParams& f, const ChunkBuffers& b,
                       int n_bins, const PassParams& pp, cudaStream_t s) {
  int blocks = (f.n_rays + kSamplerThreads - 1) / kSamplerThreads;
  int use_smem = n_bins <= 8192;
  size_t smem = use_smem ? (size_t)n_bins * sizeof(uint32_t) : 0;
  k_pass_count<<<blocks, kSamplerThreads, smem, s>>>(g, grid, f, b, n_bins, use_smem, pp);
}

void launch_export_samples(const GridParams& g, const ChunkBuffers& b, int n_bins, unsigned n_segs,
                           float* t, int32_t* subfield, cudaStream_t s) {
  if (!n_segs) return;
  k_export_samples<<<(n_segs + 255) / 256, 256, 0, s>>>(g, b, n_bins, n_segs, t, subfield);
}

void launch_export_counts(const ChunkBuffers& b, unsigned n_rays, int K, uint32_t* counts, uint32_t* offsets,
                          cudaStream_t s) {
  k_export_counts<<<(n_rays + 255) / 256, 256, 0, s>>>(b, n_rays, K, counts, offsets);
}

}  // namespace r360
