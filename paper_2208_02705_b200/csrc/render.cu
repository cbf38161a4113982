// r360 -- render orchestration behind r360_render* (host code; all compute in the kernels).
//
// A call is cut into ray chunks (r360_set_chunk_rays); a chunk is 5 kernel launches (k_count, k_scan, k_emit,
// k_mlp_*, k_composite), or one such group per pass with r360_set_wavefront.  The host never waits for the GPU
// in the middle of a frame: the kernels behind k_scan take their counts from device memory (kernels.h: totals),
// and the segment buffers (seg_td, recs, out) are sized from a CAPACITY learnt from earlier frames
// (largest segments-per-ray ratio seen, plus a quarter).  If a chunk has more segments than the capacity, k_scan
// raises kTotOverflow, the chunk's remaining kernels return at once, and the host -- which finds the flag in
// mapped pinned memory at its next call on the scene (r360_settle: r360_wait, r360_get_stats, the next render
// ...) -- renders that chunk again with larger buffers, in stream order, before anything else.  Nothing is ever
// truncated.  The very first chunk of a scene (no ratio known yet) and every retry run in the exact mode: the
// host waits for k_scan and sizes the buffers from the true count.
#include <cmath>
#include <cstring>
#include <new>

#include "scene.h"

using namespace r360;

namespace {

constexpr double kPi = 3.14159265358979323846;

// Inside a stream capture nothing may be allocated (g_no_alloc): a buffer that is too small is R360_ERR_CAPACITY.
thread_local bool g_no_alloc = false;

// Every free or reallocation of a buffer that a captured CUDA graph may have baked in (chunk buffers, tables,
// poses) bumps the scene's buffer generation: a graph captured at an older generation must not be replayed
// (r360_graph_status, r360_set_graph_poses).
template <typename T>
r360_status grow(r360_scene* sc, T*& p, size_t& cap, size_t need) {
  if (need <= cap && p) return R360_OK;
  if (g_no_alloc) return R360_ERR_CAPACITY;
  sc->buf_gen += 1;
  if (p) { cudaFree(p); p = nullptr; }           // (waits for the work that still uses it)
  const size_t want = need + 64;
  cudaError_t e = cudaMalloc(&p, want * sizeof(T));
  if (e != cudaSuccess) { cap = 0; return r360_cuda_fail(e, "cudaMalloc(chunk buffer)"); }
  cap = want;
  return R360_OK;
}

bool capturing(cudaStream_t s) {
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(s, &st) != cudaSuccess) { cudaGetLastError(); return false; }
  return st != cudaStreamCaptureStatusNone;
}

// Reading B1/B2: pixel-centre angles and their trig in binary64 libm, rounded once to binary32.
r360_status ensure_tables(r360_scene* sc, int W, int H) {
  if (sc->d_tables && sc->tab_W == W && sc->tab_H == H && sc->tab_cam_model == sc->cam_model &&
      (sc->cam_model == 0 || std::memcmp(sc->tab_cam, sc->cam, sizeof(sc->cam)) == 0))
    return R360_OK;
  if (capturing(sc->stream)) return R360_ERR_CAPACITY;   // (render this image size once before capturing)
  std::vector<float> t;
  try { t.assign((size_t)2 * W + 2 * H, 0.0f); } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
  if (sc->cam_model == 1) {
    // reading P: x_i = (i + 0.5 - cx)/fx, y_j = (j + 0.5 - cy)/fy in binary64, rounded once to binary32
    for (int i = 0; i < W; ++i) t[i] = (float)((((double)i + 0.5) - sc->cam[2]) / sc->cam[0]);
    for (int j = 0; j < H; ++j) t[(size_t)2 * W + j] = (float)((((double)j + 0.5) - sc->cam[3]) / sc->cam[1]);
  }
  for (int i = 0; i < W && sc->cam_model == 0; ++i) {
    double phi = (((double)i + 0.5) - (double)W / 2.0) * (2.0 * kPi / (double)W);
    t[i] = (float)std::sin(phi);
    t[(size_t)W + i] = (float)std::cos(phi);
  }
  for (int j = 0; j < H && sc->cam_model == 0; ++j) {
    double theta = -((((double)j + 0.5) - (double)H / 2.0) * (kPi / (double)H));
    t[(size_t)2 * W + j] = (float)std::sin(theta);
    t[(size_t)2 * W + H + j] = (float)std::cos(theta);
  }
  // earlier frames may still be reading the old tables: cudaFree waits for the device
  sc->buf_gen += 1;
  if (sc->d_tables) { cudaFree(sc->d_tables); sc->d_tables = nullptr; }
  R360_CUDA(cudaMalloc(&sc->d_tables, t.size() * sizeof(float)));
  // copy from a stack-owned vector; ordered before later work on sc->stream by a sync
  R360_CUDA(cudaMemcpyAsync(sc->d_tables, t.data(), t.size() * sizeof(float), cudaMemcpyHostToDevice, sc->stream));
  R360_CUDA(cudaStreamSynchronize(sc->stream));
  sc->tab_W = W;
  sc->tab_H = H;
  sc->tab_cam_model = sc->cam_model;
  std::memcpy(sc->tab_cam, sc->cam, sizeof(sc->cam));
  return R360_OK;
}

r360_status upload_poses(r360_scene* sc, const float* poses, int B) {
  if (!r360_poses_ok(poses, B)) return R360_ERR_INVALID_ARG;   // non-finite, or a (nearly) singular 3x3 part (B5)
  const bool cap = capturing(sc->stream);
  if (B > sc->poses_cap) {
    if (cap) return R360_ERR_CAPACITY;
    sc->buf_gen += 1;
    if (sc->d_poses) { cudaFree(sc->d_poses); sc->d_poses = nullptr; }
    if (sc->h_poses) { cudaFreeHost(sc->h_poses); sc->h_poses = nullptr; }
    sc->poses_cap = 0;
    R360_CUDA(cudaMalloc(&sc->d_poses, (size_t)B * 12 * sizeof(float)));
    R360_CUDA(cudaMallocHost(&sc->h_poses, (size_t)B * 12 * sizeof(float)));
    sc->poses_cap = B;
  }
  if (cap) {
    // inside a CUDA graph: the copy node reads the scene's pinned pose buffer at every replay, so a replay
    // renders whatever r360_set_graph_poses put there last
    std::memcpy(sc->h_poses, poses, (size_t)B * 12 * sizeof(float));
    R360_CUDA(cudaMemcpyAsync(sc->d_poses, sc->h_poses, (size_t)B * 12 * sizeof(float), cudaMemcpyHostToDevice, sc->stream));
  } else {
    // pageable source: the runtime stages it before returning, the caller may reuse `poses`
    R360_CUDA(cudaMemcpyAsync(sc->d_poses, poses, (size_t)B * 12 * sizeof(float), cudaMemcpyHostToDevice, sc->stream));
  }
  return R360_OK;
}

struct ChunkJob {
  long long ray0;        // first global ray (pose * W * H + pixel)
  unsigned n_rays;
  long long out0;        // index of that ray in the caller's output buffers
};

FrameParams frame_params(const r360_scene* sc, int W, int H, const ChunkJob& job) {
  FrameParams f;
  f.W = W; f.H = H; f.ray0 = job.ray0; f.n_rays = job.n_rays;
  f.out0 = job.out0;
  f.out_format = sc->out_format;
  f.pose0 = (unsigned)(job.ray0 / ((long long)W * H));
  f.pix0 = (unsigned)(job.ray0 % ((long long)W * H));
  f.camera = sc->cam_model;
  f.poses = sc->d_poses;
  f.sin_phi = sc->d_tables;
  f.cos_phi = sc->d_tables + W;
  f.sin_theta = sc->d_tables + 2 * (size_t)W;
  f.cos_theta = sc->d_tables + 2 * (size_t)W + H;
  return f;
}

r360_scene::ChunkEvents* chunk_events(r360_scene* sc, unsigned idx) {
  while (sc->events.size() <= idx) {
    r360_scene::ChunkEvents ce;
    for (auto& e : ce.e)
      if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    if (cudaEventCreateWithFlags(&ce.scanned, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    if (cudaEventCreateWithFlags(&ce.finished, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    try { sc->events.push_back(ce); } catch (const std::bad_alloc&) { return nullptr; }
  }
  return &sc->events[idx];
}

size_t out_bytes_per_segment(const r360_scene* sc) {
  // per-sample MLP outputs (sigma, r, g, b): float4 on the fp32 path, four binary16 values on the tensor paths
  return (size_t)sc->grid_p.K * (sc->precision >= 1 ? 8 : 16);
}

// capacity of the segment buffers, in segments
unsigned long long seg_capacity(const r360_scene* sc) {
  size_t c = sc->seg_td_cap;
  if (sc->recs_cap / kRecWords < c) c = sc->recs_cap / kRecWords;
  const size_t oc = sc->out_cap_bytes / out_bytes_per_segment(sc);
  if (oc < c) c = oc;
  if (c > 0xFFFFFFFFull) c = 0xFFFFFFFFull;                   // 32-bit segment slots
  return (unsigned long long)c;
}

// segments a chunk of n_rays rays is given room for: the largest segments-per-ray ratio seen so far + 25 %
size_t expected_segments(const r360_scene* sc, size_t n_rays) {
  return (size_t)(sc->segs_per_ray_max * 1.25 * (double)n_rays) + 4096;
}

r360_status grow_segment_buffers(r360_scene* sc, size_t n_segs) {
  r360_status st;
  if ((st = grow(sc, sc->buf.seg_td, sc->seg_td_cap, n_segs)) != R360_OK) return st;
  if ((st = grow(sc, sc->buf.recs, sc->recs_cap, n_segs * kRecWords)) != R360_OK) return st;
  unsigned char* o = reinterpret_cast<unsigned char*>(sc->buf.out);
  st = grow(sc, o, sc->out_cap_bytes, n_segs * out_bytes_per_segment(sc));
  sc->buf.out = reinterpret_cast<float4*>(o);
  return st;
}

// One chunk: steps a1-a10.  exact: wait for every k_scan and size the segment buffers from its count (first
// chunk of a scene, retries, r360_debug_samples); otherwise nothing waits for the GPU.
// sample_only: stop behind k_emit (r360_debug_samples), or behind the MLP kernel with stop_behind_mlp
// (r360_debug_field); n_segs_out then receives the segment count.
r360_status run_chunk(r360_scene* sc, int W, int H, const ChunkJob& job, unsigned chunk_idx, bool exact,
                      void* out_rgb, void* out_depth, unsigned& launches, bool sample_only = false,
                      unsigned long long* n_segs_out = nullptr, bool stop_behind_mlp = false) {
  const int n = sc->desc.n_subfields;
  const FrameParams f = frame_params(sc, W, H, job);
  const size_t n_blocks = (f.n_rays + kSamplerThreads - 1) / kSamplerThreads;
  cudaStream_t s = sc->stream;
  const bool cap = capturing(s);
  if (chunk_idx >= r360_scene::kMaxChunks) return R360_ERR_INVALID_ARG;
  r360_status st;
  struct NoAlloc {                                             // nothing is allocated inside a stream capture
    explicit NoAlloc(bool on) { g_no_alloc = on; }
    ~NoAlloc() { g_no_alloc = false; }
  } no_alloc(cap);
  if ((st = grow(sc, sc->buf.ray_cnt, sc->ray_cnt_cap, f.n_rays)) != R360_OK) return st;
  if ((st = grow(sc, sc->buf.ray_off, sc->ray_off_cap, f.n_rays)) != R360_OK) return st;
  if ((st = grow(sc, sc->buf.block_sum, sc->blocks_cap, n_blocks)) != R360_OK) return st;
  if ((st = grow(sc, sc->buf.hit_t, sc->hit_t_cap, (size_t)f.n_rays * kHitCap)) != R360_OK) return st;
  if ((st = grow(sc, sc->buf.hit_lab, sc->hit_lab_cap, (size_t)f.n_rays * kHitCap)) != R360_OK) return st;
  if (sc->precision >= 1) {            // tensor path: per-ray records (direction + packed F(d))
    if ((st = grow(sc, sc->d_dirblk, sc->dirblk_cap, (size_t)f.n_rays * 4)) != R360_OK) return st;
    sc->buf.dirblk = sc->d_dirblk;
    sc->buf.dir_f16 = sc->precision == 2;
  } else {
    sc->buf.dirblk = nullptr;
  }
  if ((st = grow(sc, sc->buf.blk_list, sc->blk_list_cap, n_blocks * kBlkListCap)) != R360_OK) return st;
  if ((st = grow(sc, sc->buf.blk_list_n, sc->blk_list_n_cap, n_blocks)) != R360_OK) return st;
  sc->buf.pass_cnt = nullptr;
  const bool wave = sc->wave_now && !sample_only;
  if (wave) {
    if ((st = grow(sc, sc->d_pass_cnt, sc->pass_cnt_cap, f.n_rays)) != R360_OK) return st;
    if ((st = grow(sc, sc->buf.pass_off, sc->pass_off_cap, f.n_rays)) != R360_OK) return st;
    if ((st = grow(sc, sc->buf.st_c, sc->st_c_cap, f.n_rays)) != R360_OK) return st;
    if ((st = grow(sc, sc->buf.st_T, sc->st_T_cap, f.n_rays)) != R360_OK) return st;
    sc->buf.pass_cnt = sc->d_pass_cnt;
  }
  if (!exact && (st = grow_segment_buffers(sc, expected_segments(sc, f.n_rays))) != R360_OK) return st;

  r360_scene::ChunkEvents* ev = chunk_events(sc, chunk_idx);
  if (!ev) return R360_ERR_OOM;
  // pinned slots of this chunk: [2c] = {overflow flag, largest pass} posted by k_scan, [2c + 1] = the counters
  unsigned long long* snap_tot = sc->h_snap + ((size_t)chunk_idx * 2 + 1) * kTotN;
  sc->buf.host_flags = sc->d_snap + (size_t)chunk_idx * 2 * kTotN;
  // single pass over all hits, or the wavefront passes (kernels.h: PassParams)
  static const uint32_t kPassEnd[5] = {2, 6, 16, (uint32_t)kHitCap, 0xFFFFFFFFu};
  const int n_pass = wave ? 5 : 1;
  for (int p = 0; p < n_pass; ++p) {
    PassParams pp{};
    if (wave) {
      pp.wavefront = 1;
      pp.first = p == 0;
      pp.last = p == n_pass - 1;
      pp.h0 = p ? kPassEnd[p - 1] : 0;
      pp.h1 = kPassEnd[p];
    }
    const bool timed = p == 0 && !cap;                         // stage times: first pass only
    // totals | bin_cnt | bin_ovf are one allocation (capi.cu): the chunk's first pass clears all of it with one
    // memset, a later wavefront pass only the two histograms
    if (p == 0) R360_CUDA(cudaMemsetAsync(sc->buf.totals, 0, kTotN * sizeof(unsigned long long) + (size_t)n * 8, s));
    else R360_CUDA(cudaMemsetAsync(sc->buf.bin_cnt, 0, (size_t)n * 8, s));
    if (timed) cudaEventRecord(ev->e[0], s);
    if (!wave || pp.first) {
      launch_count(sc->grid_p, sc->d_grid, f, sc->buf, n, s);
      launches += 1;
    }
    if (wave) {
      launch_pass_count(sc->grid_p, sc->d_grid, f, sc->buf, n, pp, s);
      launches += 1;
    }
    if (timed) cudaEventRecord(ev->e[1], s);
    launch_scan(sc->buf, (int)n_blocks, n, sc->segs_per_tile, exact ? 0xFFFFFFFFull : seg_capacity(sc),
                wave && !pp.first, s);
    if (timed) cudaEventRecord(ev->e[2], s);
    launches += 1;
    R360_CUDA(cudaGetLastError());
    if (exact) {
      R360_CUDA(cudaMemcpyAsync(snap_tot, sc->buf.totals, kTotN * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
      R360_CUDA(cudaStreamSynchronize(s));
      const unsigned long long n_segs = snap_tot[kTotSegs];
      if (snap_tot[kTotOverflow]) return R360_ERR_INVALID_ARG;   // chunk too large for 32-bit segment slots
      if (n_segs_out) *n_segs_out = n_segs;
      if (p > 0 && n_segs == 0) break;                         // every ray has finished
      double ratio = (double)n_segs / (double)f.n_rays;
      if (ratio < 1e-6) ratio = 1e-6;                          // (an empty view still ends the exact mode)
      if (ratio > sc->segs_per_ray_max) sc->segs_per_ray_max = ratio;
      // room for this count, and for what the asynchronous mode will ask for a chunk of this size
      const size_t want = expected_segments(sc, f.n_rays);
      if ((st = grow_segment_buffers(sc, want > n_segs ? want : (size_t)n_segs)) != R360_OK) return st;
    } else if (p == n_pass - 1 && !cap) {
      // k_scan has posted the chunk's overflow flag to mapped host memory; r360_settle waits for this event only
      R360_CUDA(cudaEventRecord(ev->scanned, s));
    }
    launch_emit(sc->grid_p, sc->d_grid, f, sc->buf, n, pp, s);
    launches += 1;
    R360_CUDA(cudaGetLastError());
    if (timed) cudaEventRecord(ev->e[3], s);
    if (sample_only && !stop_behind_mlp) return R360_OK;
    cudaError_t e;
    if (sc->precision >= 1)
      e = launch_mlp_tc(sc->grid_p, f, sc->buf, sc->net, sc->precision == 2 ? sc->d_wpack_f16 : sc->d_wpack,
                        sc->wpack_stride, sc->precision == 2, sc->d_frames, n, sc->segs_per_tile, sc->n_sms, s);
    else
      e = launch_mlp_fp32(sc->grid_p, f, sc->buf, sc->net, sc->lay, sc->d_wt, sc->d_frames, n, sc->segs_per_tile,
                          sc->n_sms, s);
    if (e != cudaSuccess) return r360_cuda_fail(e, "launch_mlp");
    launches += 1;
    if (sample_only) return R360_OK;
    if (timed) cudaEventRecord(ev->e[4], s);
    launch_composite(sc->grid_p, f, sc->buf, sc->desc.t_threshold, out_rgb, out_depth, pp, sc->precision >= 1, s);
    launches += 1;
    R360_CUDA(cudaGetLastError());
    if (timed) cudaEventRecord(ev->e[5], s);
  }
  // the chunk's counters for r360_get_stats
  R360_CUDA(cudaMemcpyAsync(snap_tot, sc->buf.totals, kTotN * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
  if (!cap) R360_CUDA(cudaEventRecord(ev->finished, s));
  return R360_OK;
}

void enqueue_host_copy(r360_scene* sc, const r360_scene::Pending& pd, const ChunkJob& job) {
  const size_t rgb_px = pd.out_format == 0 ? 3 * sizeof(float) : 3, d_px = pd.out_format == 0 ? sizeof(float) : 2;
  cudaEventRecord(sc->ev_chunk_done, sc->stream);
  cudaStreamWaitEvent(sc->copy_stream, sc->ev_chunk_done, 0);
  cudaMemcpyAsync((unsigned char*)pd.host_rgb + (size_t)job.out0 * rgb_px, (unsigned char*)pd.out_rgb + (size_t)job.out0 * rgb_px,
                  (size_t)job.n_rays * rgb_px, cudaMemcpyDeviceToHost, sc->copy_stream);
  cudaMemcpyAsync((unsigned char*)pd.host_depth + (size_t)job.out0 * d_px, (unsigned char*)pd.out_depth + (size_t)job.out0 * d_px,
                  (size_t)job.n_rays * d_px, cudaMemcpyDeviceToHost, sc->copy_stream);
}

}  // namespace

// The chunks enqueued by the last render call are checked: one whose segments did not fit the buffers is rendered
// again, exactly sized, in stream order.  block = false: only as far as the GPU has got (never waits).
r360_status r360_settle(r360_scene* sc, bool block) {
  r360_scene::Pending& pd = sc->pending;
  while (pd.next < pd.chunks.size()) {
    const unsigned c = pd.next;
    r360_scene::ChunkEvents& ev = sc->events[c];
    if (!block) {
      cudaError_t q = cudaEventQuery(ev.scanned);
      if (q == cudaErrorNotReady) return R360_OK;
      if (q != cudaSuccess) return r360_cuda_fail(q, "cudaEventQuery");
    } else {
      R360_CUDA(cudaEventSynchronize(ev.scanned));
    }
    const unsigned long long* snap = sc->h_snap + (size_t)c * 2 * kTotN;
    const ChunkJob job{pd.chunks[c].ray0, pd.chunks[c].n_rays, pd.chunks[c].out0};
    const double ratio = (double)snap[1] / (double)job.n_rays;           // k_scan's host_flags: {overflow, largest pass}
    if (ratio > sc->segs_per_ray_max) sc->segs_per_ray_max = ratio;
    pd.next = c + 1;
    if (snap[0]) {
      unsigned launches = 0;
      r360_status st = run_chunk(sc, pd.W, pd.H, job, c, /*exact=*/true, pd.out_rgb, pd.out_depth, launches);
      sc->stats.kernel_launches += launches;
      sc->retries += 1;
      if (st != R360_OK) { pd.chunks.clear(); pd.next = 0; return st; }
      if (pd.host_rgb) {
        enqueue_host_copy(sc, pd, job);
        if (pd.copy_done) cudaEventRecord(pd.copy_done, sc->copy_stream);
      }
    }
  }
  return R360_OK;
}

static r360_status render_device(r360_scene* sc, const float* poses, int B, int W, int H, long long ray_begin,
                                 long long ray_end, void* out_rgb, void* out_depth, void* host_rgb = nullptr,
                                 void* host_depth = nullptr, int host_bands = 1) {
  if (!sc || !poses || !out_rgb || !out_depth || B < 1 || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if ((long long)W * H >= (1ll << 30)) return R360_ERR_INVALID_ARG;
  if (ray_begin < 0 || ray_end > (long long)B * W * H || ray_begin >= ray_end) return R360_ERR_INVALID_ARG;
  r360_status st;
  const bool cap = capturing(sc->stream);
  if (!cap && (st = r360_settle(sc, true)) != R360_OK) return st;
  // inside a capture nothing can be re-rendered: chunks of the previous frame that nobody has verified yet (no
  // r360_wait before cudaStreamBeginCapture) would stay incomplete for good once this call drops them
  if (cap && sc->pending.next < sc->pending.chunks.size()) return R360_ERR_INVALID_ARG;
  if ((st = ensure_tables(sc, W, H)) != R360_OK) return st;
  if ((st = upload_poses(sc, poses, B)) != R360_OK) return st;
  const long long total_rays = ray_end - ray_begin;
  long long chunk = sc->chunk_rays < 1 ? 1 : sc->chunk_rays;
  if (chunk > (1ll << 30)) chunk = 1ll << 30;
  // host output: a call that is a single chunk is cut into bands, so that all but the last band's copy to the host
  // runs behind the next band's kernels
  if (host_rgb && host_bands > 1 && total_rays <= chunk && total_rays >= 64 * 1024 * (long long)host_bands)
    chunk = (total_rays + host_bands - 1) / host_bands;
  const long long n_chunks = (total_rays + chunk - 1) / chunk;
  if (n_chunks > (long long)r360_scene::kMaxChunks) return R360_ERR_INVALID_ARG;   // (raise r360_set_chunk_rays)
  r360_scene::Pending& pd = sc->pending;
  try {
    pd.chunks.clear();
    pd.chunks.reserve((size_t)n_chunks);
  } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
  pd.next = 0;
  pd.W = W; pd.H = H;
  pd.out_rgb = out_rgb; pd.out_depth = out_depth; pd.host_rgb = host_rgb; pd.host_depth = host_depth;
  if (!host_rgb) pd.copy_done = nullptr;
  pd.out_format = sc->out_format;
  // wavefront mode 2 (automatic): passes only if the last finished frame used less than half of its samples
  // (opaque surfaces); a translucent scene, where every sample is needed, keeps the cheaper single pass
  if (!cap && sc->chunks_last && sc->events.size() && cudaEventQuery(sc->events[0].finished) == cudaSuccess) {
    const unsigned long long* snap = sc->h_snap + kTotN;        // chunk 0 of the last call
    const unsigned long long emitted = (sc->wave_now ? snap[kTotGeo] : snap[kTotSegSum]) * (unsigned long long)sc->grid_p.K;
    if (emitted) sc->used_ratio = (double)snap[kTotUsed] / (double)emitted;
  }
  cudaGetLastError();
  if (!cap) sc->wave_now = sc->wavefront == 1 || (sc->wavefront == 2 && sc->used_ratio < 0.5);
  r360_stats& stats = sc->stats;
  std::memset(&stats, 0, sizeof(stats));
  stats.rays = (uint64_t)total_rays;
  unsigned launches = 0, chunk_idx = 0;
  for (long long r0 = 0; r0 < total_rays; r0 += chunk, ++chunk_idx) {
    const ChunkJob job{ray_begin + r0, (unsigned)((total_rays - r0 < chunk) ? (total_rays - r0) : chunk), r0};
    // the first chunk a scene ever renders sizes the buffers from its true count; everything after is asynchronous
    const bool exact = sc->segs_per_ray_max == 0.0;
    if (cap && exact) return R360_ERR_CAPACITY;                // (render once before capturing)
    if ((st = run_chunk(sc, W, H, job, chunk_idx, exact, out_rgb, out_depth, launches)) != R360_OK) {
      pd.chunks.clear();
      pd.next = 0;
      return st;
    }
    pd.chunks.push_back({job.ray0, job.n_rays, job.out0});   // (capacity reserved above: cannot throw)
    if (exact) pd.next = chunk_idx + 1;                        // nothing to verify
    if (host_rgb) enqueue_host_copy(sc, pd, job);
    if (!cap && !exact && (st = r360_settle(sc, false)) != R360_OK) return st;   // earlier chunks, without waiting
  }
  stats.chunks = chunk_idx;
  stats.kernel_launches = launches;
  sc->chunks_last = chunk_idx;
  if (cap) {                                                   // a captured frame is checked with r360_graph_status
    pd.chunks.clear();
    pd.next = 0;
    sc->graph_gen = sc->buf_gen;                               // the addresses and capacities the graph holds
    sc->graph_live = true;
  }
  return R360_OK;
}

extern "C" {

r360_status r360_render_batch(r360_scene* sc, const float* poses, int32_t B, int32_t W, int32_t H,
                              void* out_rgb, void* out_depth) {
  return render_device(sc, poses, B, W, H, 0, (long long)B * W * H, out_rgb, out_depth);
}

r360_status r360_render(r360_scene* sc, const float pose[12], int32_t W, int32_t H, void* out_rgb,
                        void* out_depth) {
  return render_device(sc, pose, 1, W, H, 0, (long long)W * H, out_rgb, out_depth);
}

r360_status r360_render_rows(r360_scene* sc, const float pose[12], int32_t W, int32_t H, int32_t row0, int32_t row1,
                             void* out_rgb, void* out_depth) {
  if (W < 1 || H < 1 || row0 < 0 || row1 > H || row0 >= row1) return R360_ERR_INVALID_ARG;
  return render_device(sc, pose, 1, W, H, (long long)row0 * W, (long long)row1 * W, out_rgb, out_depth);
}

r360_status r360_render_batch_host_async(r360_scene* sc, const float* poses, int32_t B, int32_t W, int32_t H,
                                         void* out_rgb_host, void* out_depth_host) {
  if (!sc || !poses || !out_rgb_host || !out_depth_host || B < 1 || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if (capturing(sc->stream)) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;       // (re-renders and re-copies the previous frame if needed)
  if (!sc->copy_stream) {
    R360_CUDA(cudaStreamCreateWithFlags(&sc->copy_stream, cudaStreamNonBlocking));
    R360_CUDA(cudaEventCreateWithFlags(&sc->ev_chunk_done, cudaEventDisableTiming));
    for (auto& e : sc->ev_copy_done) R360_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  }
  const int cur = sc->stage_idx ^= 1;
  const size_t R = (size_t)B * W * H;
  if (R > sc->stage_rays_cap[cur]) {
    cudaFree(sc->d_stage_rgb[cur]); cudaFree(sc->d_stage_depth[cur]);
    sc->d_stage_rgb[cur] = sc->d_stage_depth[cur] = nullptr;
    sc->stage_rays_cap[cur] = 0;
    R360_CUDA(cudaMalloc(&sc->d_stage_rgb[cur], R * 3 * sizeof(float)));
    R360_CUDA(cudaMalloc(&sc->d_stage_depth[cur], R * sizeof(float)));
    sc->stage_rays_cap[cur] = R;
  }
  // this staging set was last used two frames ago: its copy must have left before the kernels overwrite it.  A HOST
  // wait (almost always already satisfied), so that the header's promise holds: when this call returns, the frame
  // of the second-last call is in its host buffers
  R360_CUDA(cudaEventSynchronize(sc->ev_copy_done[cur]));
  sc->pending.copy_done = sc->ev_copy_done[cur];
  st = render_device(sc, poses, B, W, H, 0, (long long)R, sc->d_stage_rgb[cur], sc->d_stage_depth[cur], out_rgb_host,
                     out_depth_host, sc->host_bands);
  cudaEventRecord(sc->ev_copy_done[cur], sc->copy_stream);
  return st;
}

r360_status r360_host_sync(r360_scene* sc) {
  if (!sc) return R360_ERR_INVALID_ARG;
  // a chunk that overflowed is rendered and copied again here
  r360_status st = r360_settle(sc, true);
  // on an error too: no copy may still be writing the caller's buffers when this returns
  cudaError_t e2 = cudaStreamSynchronize(sc->stream);
  cudaError_t e1 = sc->copy_stream ? cudaStreamSynchronize(sc->copy_stream) : cudaSuccess;
  sc->pending.host_rgb = sc->pending.host_depth = nullptr;
  sc->pending.copy_done = nullptr;
  if (st != R360_OK) return st;
  if (e1 != cudaSuccess) return r360_cuda_fail(e1, "cudaStreamSynchronize(copy_stream)");
  if (e2 != cudaSuccess) return r360_cuda_fail(e2, "cudaStreamSynchronize(stream)");
  return R360_OK;
}

r360_status r360_render_batch_host(r360_scene* sc, const float* poses, int32_t B, int32_t W, int32_t H,
                                   void* out_rgb_host, void* out_depth_host) {
  r360_status st = r360_render_batch_host_async(sc, poses, B, W, H, out_rgb_host, out_depth_host);
  if (st == R360_ERR_INVALID_ARG && (!sc || !poses || !out_rgb_host || !out_depth_host || B < 1 || W < 1 || H < 1)) return st;
  r360_status st2 = sc ? r360_host_sync(sc) : R360_ERR_INVALID_ARG;
  return st != R360_OK ? st : st2;
}

r360_status r360_wait(r360_scene* sc) {
  if (!sc) return R360_ERR_INVALID_ARG;
  return r360_settle(sc, true);
}

r360_status r360_graph_status(r360_scene* sc) {
  if (!sc) return R360_ERR_INVALID_ARG;
  R360_CUDA(cudaStreamSynchronize(sc->stream));
  // a buffer the graph holds the address of was freed or reallocated by a later call outside the capture
  if (sc->graph_live && sc->graph_gen != sc->buf_gen) return R360_ERR_CAPACITY;
  for (unsigned c = 0; c < sc->chunks_last; ++c)
    if (sc->h_snap[(size_t)c * 2 * kTotN]) return R360_ERR_CAPACITY;
  return R360_OK;
}

r360_status r360_set_graph_poses(r360_scene* sc, const float* poses, int32_t B) {
  if (!sc || !poses || B < 1 || B > sc->poses_cap || !sc->h_poses) return R360_ERR_INVALID_ARG;
  if (!r360_poses_ok(poses, B)) return R360_ERR_INVALID_ARG;
  if (sc->graph_live && sc->graph_gen != sc->buf_gen) return R360_ERR_CAPACITY;   // stale graph: capture again
  std::memcpy(sc->h_poses, poses, (size_t)B * 12 * sizeof(float));
  return R360_OK;
}

r360_status r360_reserve(r360_scene* sc, uint64_t max_rays_per_chunk, double segments_per_ray) {
  if (!sc || max_rays_per_chunk < 1 || max_rays_per_chunk > (1ull << 30) || !(segments_per_ray > 0.0) ||
      !std::isfinite(segments_per_ray))
    return R360_ERR_INVALID_ARG;
  if (capturing(sc->stream)) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;
  if (segments_per_ray > sc->segs_per_ray_max) sc->segs_per_ray_max = segments_per_ray;
  return grow_segment_buffers(sc, expected_segments(sc, (size_t)max_rays_per_chunk));
}

r360_status r360_set_precision(r360_scene* sc, int32_t mode) {
  if (!sc || mode < 0 || mode > 2) return R360_ERR_INVALID_ARG;
  if (mode == 1 && !sc->d_wpack) return R360_ERR_INVALID_ARG;
  if (mode == 2 && !sc->d_wpack_f16) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;
  sc->precision = mode;
  return R360_OK;
}

r360_status r360_set_output_format(r360_scene* sc, int32_t format) {
  if (!sc || (format != R360_OUT_F32 && format != R360_OUT_RGB8_D16)) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;
  sc->out_format = format;
  return R360_OK;
}

r360_status r360_set_host_bands(r360_scene* sc, int32_t bands) {
  if (!sc || bands < 1 || bands > 64) return R360_ERR_INVALID_ARG;
  sc->host_bands = bands;
  return R360_OK;
}

r360_status r360_set_wavefront(r360_scene* sc, int32_t mode) {
  if (!sc || mode < 0 || mode > 2) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;
  sc->wavefront = mode;
  sc->wave_now = mode == 1;
  sc->used_ratio = 1.0;
  return R360_OK;
}

r360_status r360_set_camera(r360_scene* sc, int32_t model, double fx, double fy, double cx, double cy) {
  if (!sc || (model != 0 && model != 1)) return R360_ERR_INVALID_ARG;
  if (model == 1 && !(fx > 0.0 && fy > 0.0 && std::isfinite(fx) && std::isfinite(fy) && std::isfinite(cx) &&
                      std::isfinite(cy)))
    return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;
  sc->cam_model = model;
  sc->cam[0] = fx; sc->cam[1] = fy; sc->cam[2] = cx; sc->cam[3] = cy;
  return R360_OK;
}

r360_status r360_set_stream(r360_scene* sc, void* stream) {
  if (!sc) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;
  if ((cudaStream_t)stream != sc->stream) {
    // work of earlier calls on the old stream shares the scene's buffers with what follows on the new one
    // (the caller may already have destroyed the old stream: its work is complete then, the error is dropped)
    if (cudaStreamSynchronize(sc->stream) != cudaSuccess) cudaGetLastError();
  }
  sc->stream = (cudaStream_t)stream;
  return R360_OK;
}

r360_status r360_set_chunk_rays(r360_scene* sc, int64_t max_rays) {
  if (!sc || max_rays < 1) return R360_ERR_INVALID_ARG;
  sc->chunk_rays = max_rays;
  return R360_OK;
}

r360_status r360_get_stats(r360_scene* sc, r360_stats* out) {
  if (!sc || !out) return R360_ERR_INVALID_ARG;
  r360_status rs;
  if ((rs = r360_settle(sc, true)) != R360_OK) return rs;
  R360_CUDA(cudaStreamSynchronize(sc->stream));
  r360_stats& st = sc->stats;
  st.ms_count = st.ms_scan = st.ms_emit = st.ms_mlp = st.ms_composite = st.ms_total = 0.f;
  st.segments = st.mlp_tiles = st.samples_used = st.samples_emitted = 0;
  for (unsigned c = 0; c < sc->chunks_last && c < sc->events.size(); ++c) {
    float ms[5] = {0, 0, 0, 0, 0};
    for (int i = 0; i < 5; ++i)
      if (cudaEventElapsedTime(&ms[i], sc->events[c].e[i], sc->events[c].e[i + 1]) != cudaSuccess) ms[i] = 0.f;
    st.ms_count += ms[0]; st.ms_scan += ms[1]; st.ms_emit += ms[2]; st.ms_mlp += ms[3]; st.ms_composite += ms[4];
    const unsigned long long* snap = sc->h_snap + ((size_t)c * 2 + 1) * kTotN;
    st.segments += snap[kTotSegSum];
    st.mlp_tiles += snap[kTotTileSum];
    st.samples_used += snap[kTotUsed];
    // wavefront: `segments` counts what reached the MLP; the geometric total comes from the walk
    st.samples_emitted += (sc->wave_now ? snap[kTotGeo] : snap[kTotSegSum]) * (uint64_t)sc->grid_p.K;
  }
  cudaGetLastError();
  st.ms_total = st.ms_count + st.ms_scan + st.ms_emit + st.ms_mlp + st.ms_composite;
  st.retries = sc->retries;
  *out = st;
  return R360_OK;
}

static r360_status debug_tap(r360_scene* sc, const float pose[12], int32_t W, int32_t H, uint32_t* counts,
                             uint32_t* offsets, float* t, int32_t* subfield, float* field, bool with_field,
                             uint64_t cap, uint64_t* total);

r360_status r360_debug_samples(r360_scene* sc, const float pose[12], int32_t W, int32_t H, uint32_t* counts,
                               uint32_t* offsets, float* t, int32_t* subfield, uint64_t cap, uint64_t* total) {
  return debug_tap(sc, pose, W, H, counts, offsets, t, subfield, nullptr, false, cap, total);
}

r360_status r360_debug_field(r360_scene* sc, const float pose[12], int32_t W, int32_t H, uint32_t* counts,
                             uint32_t* offsets, float* t, int32_t* subfield, float* field, uint64_t cap,
                             uint64_t* total) {
  return debug_tap(sc, pose, W, H, counts, offsets, t, subfield, field, true, cap, total);
}

}  // extern "C"

static r360_status debug_tap(r360_scene* sc, const float pose[12], int32_t W, int32_t H, uint32_t* counts,
                             uint32_t* offsets, float* t, int32_t* subfield, float* field, bool with_field,
                             uint64_t cap, uint64_t* total) {
  if (!sc || !pose || !counts || !offsets || !total || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if ((long long)W * H >= (1ll << 30)) return R360_ERR_INVALID_ARG;
  if (capturing(sc->stream)) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = r360_settle(sc, true)) != R360_OK) return st;
  if ((st = ensure_tables(sc, W, H)) != R360_OK) return st;
  if ((st = upload_poses(sc, pose, 1)) != R360_OK) return st;
  const ChunkJob job{0, (unsigned)((long long)W * H), 0};
  unsigned long long n_segs = 0;
  unsigned launches = 0;
  if ((st = run_chunk(sc, W, H, job, 0, /*exact=*/true, nullptr, nullptr, launches, /*sample_only=*/true, &n_segs,
                      /*stop_behind_mlp=*/with_field)) != R360_OK)
    return st;
  sc->chunks_last = 0;
  *total = n_segs * (uint64_t)sc->grid_p.K;
  launch_export_counts(sc->buf, job.n_rays, sc->grid_p.K, counts, offsets, sc->stream);
  R360_CUDA(cudaGetLastError());
  if (*total > cap) { cudaStreamSynchronize(sc->stream); return R360_ERR_CAPACITY; }
  if (n_segs) {
    if (!t || !subfield || (with_field && !field)) return R360_ERR_INVALID_ARG;
    launch_export_samples(sc->grid_p, sc->buf, sc->desc.n_subfields, (unsigned)n_segs, t, subfield, sc->stream);
    if (with_field) launch_export_field(sc->buf, (size_t)n_segs * sc->grid_p.K, sc->precision >= 1, field, sc->stream);
    R360_CUDA(cudaGetLastError());
  }
  R360_CUDA(cudaStreamSynchronize(sc->stream));
  return R360_OK;
}
