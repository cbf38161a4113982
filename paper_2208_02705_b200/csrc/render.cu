// r360 -- render orchestration behind r360_render* (host code; all compute in the kernels).
#include <cmath>
#include <cstring>

#include "scene.h"

using namespace r360;

namespace {

constexpr double kPi = 3.14159265358979323846;

template <typename T>
r360_status grow(T*& p, size_t& cap, size_t need, size_t slack_num = 5, size_t slack_den = 4) {
  if (need <= cap && p) return R360_OK;
  if (p) { cudaFree(p); p = nullptr; }
  size_t want = need * slack_num / slack_den + 64;
  cudaError_t e = cudaMalloc(&p, want * sizeof(T));
  if (e != cudaSuccess) { cap = 0; return r360_cuda_fail(e, "cudaMalloc(chunk buffer)"); }
  cap = want;
  return R360_OK;
}

// Reading B1/B2: pixel-centre angles and their trig in binary64 libm, rounded once to binary32.
r360_status ensure_tables(r360_scene* sc, int W, int H) {
  if (sc->d_tables && sc->tab_W == W && sc->tab_H == H && sc->tab_cam_model == sc->cam_model &&
      (sc->cam_model == 0 || std::memcmp(sc->tab_cam, sc->cam, sizeof(sc->cam)) == 0))
    return R360_OK;
  std::vector<float> t((size_t)2 * W + 2 * H, 0.0f);
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
  if (sc->d_tables) { cudaFree(sc->d_tables); sc->d_tables = nullptr; }
  R360_CUDA(cudaMalloc(&sc->d_tables, t.size() * sizeof(float)));
  // synchronous copy from a stack-owned vector; ordered before later work on sc->stream by a sync
  R360_CUDA(cudaMemcpyAsync(sc->d_tables, t.data(), t.size() * sizeof(float), cudaMemcpyHostToDevice, sc->stream));
  R360_CUDA(cudaStreamSynchronize(sc->stream));
  sc->tab_W = W;
  sc->tab_H = H;
  sc->tab_cam_model = sc->cam_model;
  std::memcpy(sc->tab_cam, sc->cam, sizeof(sc->cam));
  return R360_OK;
}

r360_status upload_poses(r360_scene* sc, const float* poses, int B) {
  for (int i = 0; i < B * 12; ++i)
    if (!std::isfinite(poses[i])) return R360_ERR_INVALID_ARG;
  if (B > sc->poses_cap) {
    if (sc->d_poses) { cudaFree(sc->d_poses); sc->d_poses = nullptr; }
    R360_CUDA(cudaMalloc(&sc->d_poses, (size_t)B * 12 * sizeof(float)));
    sc->poses_cap = B;
  }
  // pageable source: the runtime stages it before returning, the caller may reuse `poses`
  R360_CUDA(cudaMemcpyAsync(sc->d_poses, poses, (size_t)B * 12 * sizeof(float), cudaMemcpyHostToDevice, sc->stream));
  return R360_OK;
}

FrameParams frame_params(const r360_scene* sc, int W, int H, long long ray0, unsigned n_rays) {
  FrameParams f;
  f.W = W; f.H = H; f.ray0 = ray0; f.n_rays = n_rays;
  f.pose0 = (unsigned)(ray0 / ((long long)W * H));
  f.pix0 = (unsigned)(ray0 % ((long long)W * H));
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
    sc->events.push_back(ce);
  }
  return &sc->events[idx];
}

// Steps a1-a5 for one chunk: count, scan, (sync for the segment total), emit.  pp.wavefront: one pass of the
// wavefronted path -- the walk (k_count) runs with the first pass only, every pass bins its own hit range.
r360_status sample_chunk(r360_scene* sc, const FrameParams& f, r360_scene::ChunkEvents* ev,
                         unsigned long long& n_segs, unsigned long long& n_tiles, unsigned& launches,
                         const PassParams& pp) {
  const int n = sc->desc.n_subfields;
  const size_t n_blocks = (f.n_rays + kSamplerThreads - 1) / kSamplerThreads;
  r360_status st;
  if ((st = grow(sc->buf.ray_cnt, sc->ray_cnt_cap, f.n_rays, 1, 1)) != R360_OK) return st;
  if ((st = grow(sc->buf.ray_off, sc->ray_off_cap, f.n_rays, 1, 1)) != R360_OK) return st;
  if ((st = grow(sc->buf.block_sum, sc->blocks_cap, n_blocks, 1, 1)) != R360_OK) return st;
  if ((st = grow(sc->buf.hit_t, sc->hit_t_cap, (size_t)f.n_rays * kHitCap, 1, 1)) != R360_OK) return st;
  if ((st = grow(sc->buf.hit_lab, sc->hit_lab_cap, (size_t)f.n_rays * kHitCap, 1, 1)) != R360_OK) return st;
  if (sc->precision >= 1) {            // tensor path: per-ray records (direction + packed F(d))
    if ((st = grow(sc->d_dirblk, sc->dirblk_cap, (size_t)f.n_rays * 4, 1, 1)) != R360_OK) return st;
    sc->buf.dirblk = sc->d_dirblk;
    sc->buf.dir_f16 = sc->precision == 2;
  } else {
    sc->buf.dirblk = nullptr;
  }
  cudaStream_t s = sc->stream;
  if ((st = grow(sc->buf.blk_list, sc->blk_list_cap, n_blocks * kBlkListCap, 1, 1)) != R360_OK) return st;
  if ((st = grow(sc->buf.blk_list_n, sc->blk_list_n_cap, n_blocks, 1, 1)) != R360_OK) return st;
  sc->buf.pass_cnt = nullptr;
  if (pp.wavefront) {
    if ((st = grow(sc->d_pass_cnt, sc->pass_cnt_cap, f.n_rays, 1, 1)) != R360_OK) return st;
    if ((st = grow(sc->buf.pass_off, sc->pass_off_cap, f.n_rays, 1, 1)) != R360_OK) return st;
    if ((st = grow(sc->buf.st_c, sc->st_c_cap, f.n_rays, 1, 1)) != R360_OK) return st;
    if ((st = grow(sc->buf.st_T, sc->st_T_cap, f.n_rays, 1, 1)) != R360_OK) return st;
    sc->buf.pass_cnt = sc->d_pass_cnt;
  }
  R360_CUDA(cudaMemsetAsync(sc->buf.bin_cnt, 0, (size_t)n * 4, s));
  R360_CUDA(cudaMemsetAsync(sc->buf.bin_ovf, 0, (size_t)n * 4, s));
  if (ev) cudaEventRecord(ev->e[0], s);
  if (!pp.wavefront || pp.first) {
    launch_count(sc->grid_p, sc->d_grid, f, sc->buf, n, s);
    launches += 1;
  }
  if (pp.wavefront) {
    launch_pass_count(sc->grid_p, sc->d_grid, f, sc->buf, n, pp, s);
    launches += 1;
  }
  if (ev) cudaEventRecord(ev->e[1], s);
  launch_scan(sc->buf, (int)n_blocks, n, sc->segs_per_tile, s);
  if (ev) cudaEventRecord(ev->e[2], s);
  launches += 1;
  R360_CUDA(cudaGetLastError());
  R360_CUDA(cudaMemcpyAsync(sc->h_totals, sc->buf.totals, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
  R360_CUDA(cudaStreamSynchronize(s));
  n_segs = sc->h_totals[0];
  n_tiles = sc->h_totals[1];
  if (n_segs >= (1ull << 32)) return R360_ERR_INVALID_ARG;   // chunk too large for 32-bit slots
  if (n_segs) {
    if ((st = grow(sc->buf.seg_tin, sc->seg_tin_cap, n_segs)) != R360_OK) return st;
    if ((st = grow(sc->buf.seg_dt, sc->seg_dt_cap, n_segs)) != R360_OK) return st;
    if ((st = grow(sc->buf.recs, sc->recs_cap, n_segs * kRecWords)) != R360_OK) return st;
    launch_emit(sc->grid_p, sc->d_grid, f, sc->buf, n, pp, s);
    launches += 1;
    R360_CUDA(cudaGetLastError());
  }
  if (ev) cudaEventRecord(ev->e[3], s);
  return R360_OK;
}

}  // namespace

// host_rgb / host_depth (both or neither): every chunk's part of the image is copied to host memory on a second
// stream as soon as the chunk is composited, behind the next chunk's kernels (r360_render_batch_host)
static r360_status render_device(r360_scene* sc, const float* poses, int B, int W, int H, float* out_rgb,
                                 float* out_depth, float* host_rgb = nullptr, float* host_depth = nullptr) {
  if (!sc || !poses || !out_rgb || !out_depth || B < 1 || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if ((long long)W * H >= (1ll << 30)) return R360_ERR_INVALID_ARG;
  const long long total_rays = (long long)B * W * H;
  r360_status st;
  if ((st = ensure_tables(sc, W, H)) != R360_OK) return st;
  if ((st = upload_poses(sc, poses, B)) != R360_OK) return st;
  cudaStream_t s = sc->stream;
  R360_CUDA(cudaMemsetAsync(sc->buf.totals, 0, 4 * sizeof(unsigned long long), s));
  r360_stats& stats = sc->stats;
  std::memset(&stats, 0, sizeof(stats));
  stats.rays = (uint64_t)total_rays;
  unsigned launches = 0, chunk_idx = 0;
  long long chunk = sc->chunk_rays < 1 ? 1 : sc->chunk_rays;
  if (chunk > (1ll << 30)) chunk = 1ll << 30;
  for (long long ray0 = 0; ray0 < total_rays; ray0 += chunk, ++chunk_idx) {
    unsigned n_rays = (unsigned)((total_rays - ray0 < chunk) ? (total_rays - ray0) : chunk);
    FrameParams f = frame_params(sc, W, H, ray0, n_rays);
    r360_scene::ChunkEvents* ev = chunk_events(sc, chunk_idx);
    // single pass over all hits, or the wavefront passes (kernels.h: PassParams)
    static const uint32_t kPassEnd[5] = {2, 6, 16, (uint32_t)kHitCap, 0xFFFFFFFFu};
    const int n_pass = sc->wavefront ? 5 : 1;
    for (int p = 0; p < n_pass; ++p) {
      PassParams pp{};
      if (sc->wavefront) {
        pp.wavefront = 1;
        pp.first = p == 0;
        pp.last = p == n_pass - 1;
        pp.h0 = p ? kPassEnd[p - 1] : 0;
        pp.h1 = kPassEnd[p];
      }
      r360_scene::ChunkEvents* pev = p == 0 ? ev : nullptr;   // stage times: first pass only
      unsigned long long n_segs = 0, n_tiles = 0;
      if ((st = sample_chunk(sc, f, pev, n_segs, n_tiles, launches, pp)) != R360_OK) return st;
      if (p > 0 && n_segs == 0) break;                       // every ray has finished
      if (n_segs) {
        // per-sample MLP outputs: K * segments float4, ray-major
        if ((st = grow(sc->buf.out, sc->out_cap, (size_t)n_segs * sc->grid_p.K)) != R360_OK) return st;
        cudaError_t e;
        if (sc->precision >= 1)
          e = launch_mlp_tc(sc->grid_p, f, sc->buf, sc->net, sc->precision == 2 ? sc->d_wpack_f16 : sc->d_wpack,
                            sc->wpack_stride, sc->precision == 2, sc->d_frames, sc->desc.n_subfields,
                            sc->segs_per_tile, sc->n_sms, s);
        else
          e = launch_mlp_fp32(sc->grid_p, f, sc->buf, sc->net, sc->lay, sc->d_wt, sc->d_frames,
                              sc->desc.n_subfields, sc->segs_per_tile, sc->n_sms, s);
        if (e != cudaSuccess) return r360_cuda_fail(e, "launch_mlp");
        launches += 1;
      }
      if (pev) cudaEventRecord(pev->e[4], s);
      launch_composite(sc->grid_p, f, sc->buf, sc->desc.t_threshold, out_rgb, out_depth, pp, sc->precision >= 1, s);
      launches += 1;
      R360_CUDA(cudaGetLastError());
      if (pev) cudaEventRecord(pev->e[5], s);
      stats.segments += n_segs;
      stats.mlp_tiles += n_tiles;
    }
    if (host_rgb) {
      R360_CUDA(cudaEventRecord(sc->ev_chunk_done, s));
      R360_CUDA(cudaStreamWaitEvent(sc->copy_stream, sc->ev_chunk_done, 0));
      R360_CUDA(cudaMemcpyAsync(host_rgb + (size_t)ray0 * 3, out_rgb + (size_t)ray0 * 3, (size_t)n_rays * 3 * sizeof(float),
                                cudaMemcpyDeviceToHost, sc->copy_stream));
      R360_CUDA(cudaMemcpyAsync(host_depth + (size_t)ray0, out_depth + (size_t)ray0, (size_t)n_rays * sizeof(float),
                                cudaMemcpyDeviceToHost, sc->copy_stream));
    }
  }
  // wavefront: `segments` counts what reached the MLP; the geometric total comes from the walk
  stats.samples_emitted = (sc->wavefront ? (uint64_t)sc->h_totals[3] : stats.segments) * (uint64_t)sc->grid_p.K;
  stats.chunks = chunk_idx;
  stats.kernel_launches = launches;
  sc->chunks_last = chunk_idx;
  return R360_OK;
}

extern "C" {

r360_status r360_render_batch(r360_scene* sc, const float* poses, int32_t B, int32_t W, int32_t H,
                              float* out_rgb, float* out_depth) {
  return render_device(sc, poses, B, W, H, out_rgb, out_depth);
}

r360_status r360_render(r360_scene* sc, const float pose[12], int32_t W, int32_t H, float* out_rgb,
                        float* out_depth) {
  return render_device(sc, pose, 1, W, H, out_rgb, out_depth);
}

r360_status r360_render_batch_host(r360_scene* sc, const float* poses, int32_t B, int32_t W, int32_t H,
                                   float* out_rgb_host, float* out_depth_host) {
  if (!sc || !poses || !out_rgb_host || !out_depth_host || B < 1 || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  const size_t R = (size_t)B * W * H;
  if (R > sc->stage_rays_cap) {
    cudaFree(sc->d_stage_rgb); cudaFree(sc->d_stage_depth);
    sc->d_stage_rgb = sc->d_stage_depth = nullptr;
    sc->stage_rays_cap = 0;
    R360_CUDA(cudaMalloc(&sc->d_stage_rgb, R * 3 * sizeof(float)));
    R360_CUDA(cudaMalloc(&sc->d_stage_depth, R * sizeof(float)));
    sc->stage_rays_cap = R;
  }
  if (!sc->copy_stream) {
    R360_CUDA(cudaStreamCreateWithFlags(&sc->copy_stream, cudaStreamNonBlocking));
    R360_CUDA(cudaEventCreateWithFlags(&sc->ev_chunk_done, cudaEventDisableTiming));
  }
  r360_status st = render_device(sc, poses, B, W, H, sc->d_stage_rgb, sc->d_stage_depth, out_rgb_host, out_depth_host);
  // on an error too: no copy may still be writing the caller's buffers when this returns
  cudaError_t e1 = cudaStreamSynchronize(sc->copy_stream), e2 = cudaStreamSynchronize(sc->stream);
  if (st != R360_OK) return st;
  if (e1 != cudaSuccess) return r360_cuda_fail(e1, "cudaStreamSynchronize(copy_stream)");
  if (e2 != cudaSuccess) return r360_cuda_fail(e2, "cudaStreamSynchronize(stream)");
  return R360_OK;
}

r360_status r360_set_precision(r360_scene* sc, int32_t mode) {
  if (!sc || mode < 0 || mode > 2) return R360_ERR_INVALID_ARG;
  if (mode == 1 && !sc->d_wpack) return R360_ERR_INVALID_ARG;
  if (mode == 2 && !sc->d_wpack_f16) return R360_ERR_INVALID_ARG;
  sc->precision = mode;
  return R360_OK;
}

r360_status r360_set_wavefront(r360_scene* sc, int32_t enable) {
  if (!sc || (enable != 0 && enable != 1)) return R360_ERR_INVALID_ARG;
  sc->wavefront = enable;
  return R360_OK;
}

r360_status r360_set_camera(r360_scene* sc, int32_t model, double fx, double fy, double cx, double cy) {
  if (!sc || (model != 0 && model != 1)) return R360_ERR_INVALID_ARG;
  if (model == 1 && !(fx > 0.0 && fy > 0.0 && std::isfinite(fx) && std::isfinite(fy) && std::isfinite(cx) &&
                      std::isfinite(cy)))
    return R360_ERR_INVALID_ARG;
  sc->cam_model = model;
  sc->cam[0] = fx; sc->cam[1] = fy; sc->cam[2] = cx; sc->cam[3] = cy;
  return R360_OK;
}

r360_status r360_set_stream(r360_scene* sc, void* stream) {
  if (!sc) return R360_ERR_INVALID_ARG;
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
  R360_CUDA(cudaStreamSynchronize(sc->stream));
  r360_stats& st = sc->stats;
  st.ms_count = st.ms_scan = st.ms_emit = st.ms_mlp = st.ms_composite = st.ms_total = 0.f;
  for (unsigned c = 0; c < sc->chunks_last && c < sc->events.size(); ++c) {
    float ms[5] = {0, 0, 0, 0, 0};
    for (int i = 0; i < 5; ++i)
      if (cudaEventElapsedTime(&ms[i], sc->events[c].e[i], sc->events[c].e[i + 1]) != cudaSuccess) ms[i] = 0.f;
    st.ms_count += ms[0]; st.ms_scan += ms[1]; st.ms_emit += ms[2]; st.ms_mlp += ms[3]; st.ms_composite += ms[4];
  }
  cudaGetLastError();
  st.ms_total = st.ms_count + st.ms_scan + st.ms_emit + st.ms_mlp + st.ms_composite;
  if (sc->chunks_last) {
    unsigned long long used = 0;
    R360_CUDA(cudaMemcpy(&used, sc->buf.totals + 2, sizeof(used), cudaMemcpyDeviceToHost));
    st.samples_used = used;
  }
  *out = st;
  return R360_OK;
}

r360_status r360_debug_samples(r360_scene* sc, const float pose[12], int32_t W, int32_t H, uint32_t* counts,
                               uint32_t* offsets, float* t, int32_t* subfield, uint64_t cap, uint64_t* total) {
  if (!sc || !pose || !counts || !offsets || !total || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if ((long long)W * H >= (1ll << 30)) return R360_ERR_INVALID_ARG;
  r360_status st;
  if ((st = ensure_tables(sc, W, H)) != R360_OK) return st;
  if ((st = upload_poses(sc, pose, 1)) != R360_OK) return st;
  FrameParams f = frame_params(sc, W, H, 0, (unsigned)((long long)W * H));
  unsigned long long n_segs = 0, n_tiles = 0;
  unsigned launches = 0;
  if ((st = sample_chunk(sc, f, nullptr, n_segs, n_tiles, launches, PassParams{})) != R360_OK) return st;
  *total = n_segs * (uint64_t)sc->grid_p.K;
  launch_export_counts(sc->buf, f.n_rays, sc->grid_p.K, counts, offsets, sc->stream);
  R360_CUDA(cudaGetLastError());
  if (*total > cap) { cudaStreamSynchronize(sc->stream); return R360_ERR_CAPACITY; }
  if (n_segs) {
    if (!t || !subfield) return R360_ERR_INVALID_ARG;
    launch_export_samples(sc->grid_p, sc->buf, sc->desc.n_subfields, (unsigned)n_segs, t, subfield, sc->stream);
    R360_CUDA(cudaGetLastError());
  }
  R360_CUDA(cudaStreamSynchronize(sc->stream));
  return R360_OK;
}

}  // extern "C"
