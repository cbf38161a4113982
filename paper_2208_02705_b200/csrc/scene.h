// r360 -- host-side scene object behind the opaque r360_scene handle.
#pragma once
#include <vector>

#include "../../include/r360.h"
#include "kernels.h"

struct r360_scene {
  r360_scene_desc desc;
  r360::GridParams grid_p;
  r360::NetShape net;
  r360::Fp32Layout lay;
  int n_sms = 148;
  int segs_per_tile = 16;
  // scene-constant device data
  uint16_t* d_grid = nullptr;               // fused occupancy + label (common.cuh)
  uint8_t* d_skip = nullptr;                // [N][8] octant skip distances of the empty voxels (common.cuh)
  r360::SubfieldFrame* d_frames = nullptr;  // [n]
  float* d_wt = nullptr;                    // [n * lay.total] fp32, transposed + padded
  void* d_wpack = nullptr;                  // [n * wpack_stride] bfloat16 operand tiles + fp32 head biases
  void* d_wpack_f16 = nullptr;              // the same in binary16; null if a weight does not fit binary16
  size_t wpack_stride = 0;
  bool tc_fits = false;                     // the tensor kernel's shared memory fits this network
  // per (W,H): trig tables; per call: poses
  float* d_tables = nullptr;
  int tab_W = 0, tab_H = 0;
  // camera (r360_set_camera): 0 equirect, 1 pinhole; tab_cam = what d_tables was built for
  int cam_model = 0;
  double cam[4] = {0, 0, 0, 0};             // fx, fy, cx, cy
  int tab_cam_model = -1;
  double tab_cam[4] = {0, 0, 0, 0};
  float* d_poses = nullptr;
  float* h_poses = nullptr;                 // pinned; source of the pose copy inside a captured CUDA graph
  int poses_cap = 0;
  // chunk buffers and capacities
  unsigned long long buf_gen = 0;           // bumped whenever a device buffer is freed or reallocated
  unsigned long long graph_gen = 0;         // buf_gen at the last captured render call
  bool graph_live = false;                  // a render call has been captured on this scene
  r360::ChunkBuffers buf{};
  size_t ray_cnt_cap = 0, ray_off_cap = 0, blocks_cap = 0;
  size_t seg_td_cap = 0, recs_cap = 0, out_cap_bytes = 0, dirblk_cap = 0, hit_t_cap = 0, hit_lab_cap = 0, blk_list_cap = 0, blk_list_n_cap = 0;
  uint4* d_dirblk = nullptr;                // owned; buf.dirblk points here only while the tensor path is selected
  // pinned, mapped snapshots of the device counters, kMaxChunks x 2 x kTotN: [2c] = what k_scan posts for chunk c
  // (overflow flag, largest pass), [2c + 1] = the counters at the end of the chunk (statistics)
  static constexpr unsigned kMaxChunks = 4096;
  unsigned long long* h_snap = nullptr;
  unsigned long long* d_snap = nullptr;     // the same memory as the device sees it
  double segs_per_ray_max = 0.0;            // largest segments-per-ray ratio of any chunk pass so far: sizes the buffers
  unsigned retries = 0;                     // chunks rendered again because their segments exceeded the capacity
  // D2H staging for r360_render_batch_host
  // two sets, used in turn: the copy of frame k runs behind the kernels of frame k+1 (r360_render_batch_host_async)
  float* d_stage_rgb[2] = {nullptr, nullptr};
  float* d_stage_depth[2] = {nullptr, nullptr};
  size_t stage_rays_cap[2] = {0, 0};
  cudaEvent_t ev_copy_done[2] = {nullptr, nullptr};   // recorded on copy_stream behind a frame's last copy
  int stage_idx = 0;
  cudaStream_t copy_stream = nullptr;       // chunk k's image part goes to the host behind chunk k+1's kernels
  cudaEvent_t ev_chunk_done = nullptr;
  // configuration
  cudaStream_t stream = nullptr;
  int precision = 0;                        // 0 fp32 ALUs, 1 tensor cores bfloat16, 2 tensor cores binary16
  int out_format = 0;                       // r360_output_format
  int host_bands = 1;                       // r360_render_batch_host cuts a single-chunk call into this many bands
  bool wave_now = false;                    // what the current / last render call does
  double used_ratio = 1.0;                  // samples composited / samples emitted of the last finished frame
  int wavefront = 0;                        // r360_set_wavefront: feed the MLP in passes, retire finished rays between them
  uint32_t* d_pass_cnt = nullptr;           // owned; buf.pass_cnt points here only during wavefront passes
  size_t pass_cnt_cap = 0, pass_off_cap = 0, st_c_cap = 0, st_T_cap = 0;
  long long chunk_rays = 4ll << 20;
  // statistics of the last call
  struct ChunkEvents { cudaEvent_t e[6]; cudaEvent_t scanned; cudaEvent_t finished; };
  std::vector<ChunkEvents> events;   // pool, one set per chunk
  unsigned chunks_last = 0;
  // the chunks enqueued by the last render call, until r360_settle has seen their overflow flags
  struct PendingChunk { long long ray0; unsigned n_rays; long long out0; };
  struct Pending {
    std::vector<PendingChunk> chunks;
    unsigned next = 0;                      // first chunk not yet verified
    int W = 0, H = 0, out_format = 0;
    void *out_rgb = nullptr, *out_depth = nullptr, *host_rgb = nullptr, *host_depth = nullptr;
    cudaEvent_t copy_done = nullptr;        // host output: re-recorded behind the copy of a re-rendered chunk
  } pending;
  r360_stats stats{};
};

// render.cu: verify the chunks of the last render call, re-render what overflowed (block: wait for their k_scan)
r360_status r360_settle(r360_scene* sc, bool block);

// capi.cu: reading B5 -- finite, and every 3x3 part well conditioned (no unit direction is mapped to ~zero)
bool r360_poses_ok(const float* poses, int B);

// records the CUDA error text for r360_last_cuda_error() and maps it to a status
r360_status r360_cuda_fail(cudaError_t e, const char* what);

#define R360_CUDA(call)                                         \
  do {                                                          \
    cudaError_t e_ = (call);                                    \
    if (e_ != cudaSuccess) return r360_cuda_fail(e_, #call);    \
  } while (0)
