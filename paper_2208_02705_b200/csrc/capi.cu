// r360 -- C ABI (include/r360.h): argument checks, scene upload, render orchestration.
// Host code only; every step of the path runs in the CUDA kernels of this directory.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>
#include <thread>
#include <vector>

#include "scene.h"

using namespace r360;

namespace {

thread_local char g_cuda_err[256] = "";

int pe_dim(int L) { return 3 + 6 * L; }

bool desc_ok(const r360_scene_desc* d) {
  if (!d) return false;
  for (int a = 0; a < 3; ++a) {
    if (d->dims[a] < 1) return false;
    if (!std::isfinite(d->box_min[a]) || !std::isfinite(d->box_max[a])) return false;
    if (!(d->box_max[a] > d->box_min[a])) return false;
  }
  if ((long long)d->dims[0] * d->dims[1] * d->dims[2] > (1ll << 31) - 1) return false;
  if (d->n_subfields < 1 || d->n_subfields > kMaxSubfields) return false;
  if (d->hidden_width != 32 && d->hidden_width != 64) return false;
  if (d->n_hidden < 1 || d->n_hidden > 8) return false;
  if (d->pe_pos_levels < 0 || d->pe_pos_levels > 16) return false;
  if (d->pe_dir_levels < 0 || d->pe_dir_levels > 8) return false;
  if (d->samples_per_voxel < 1 || d->samples_per_voxel > kTileRows) return false;
  if (!(d->t_threshold >= 0.0f) || !std::isfinite(d->t_threshold)) return false;
  if (d->density_activation != 0 && d->density_activation != 1) return false;
  if (d->occ_threshold < 1) return false;
  return true;
}

// Source blob offsets (include/r360.h order) and the padded, transposed device layout.
struct SrcLayout {
  int trunk[8], dens, feat, col, rgb, total;
};

void make_layouts(const r360_scene_desc& d, SrcLayout& s, Fp32Layout& t) {
  const int Wd = d.hidden_width, pp = pe_dim(d.pe_pos_levels), pd = pe_dim(d.pe_dir_levels);
  int so = 0, to = 0;
  auto pad4 = [](int x) { return (x + 3) & ~3; };
  for (int l = 0; l < d.n_hidden; ++l) {
    int in = l == 0 ? pp : Wd;
    s.trunk[l] = so; so += Wd * in + Wd;
    t.trunk[l] = to; to += pad4(Wd * in + Wd);
  }
  s.dens = so; so += Wd + 1;
  t.dens = to; to += pad4(Wd + 1);
  s.feat = so; so += Wd * Wd + Wd;
  t.feat = to; to += pad4(Wd * Wd + Wd);
  s.col = so; so += Wd * (Wd + pd) + Wd;
  t.col = to; to += pad4(Wd * (Wd + pd) + Wd);
  s.rgb = so; so += 3 * Wd + 3;
  t.rgb = to; to += 4 * Wd + 4;
  s.total = so;
  t.total = to;
}

// W[out][in] + b[out]  ->  W^T[in][out_pad] + b[out_pad]
void transpose_layer(const float* src, float* dst, int out, int in, int out_pad) {
  for (int i = 0; i < in; ++i)
    for (int o = 0; o < out_pad; ++o) dst[(size_t)i * out_pad + o] = o < out ? src[(size_t)o * in + i] : 0.0f;
  for (int o = 0; o < out_pad; ++o) dst[(size_t)in * out_pad + o] = o < out ? src[(size_t)out * in + o] : 0.0f;
}

}  // namespace

// DESIGN.md reading B5: B poses are admissible iff every entry is finite and every 3x3 part R (binary64) satisfies
// 2^-16 <= ||R||_F <= 2^16 and |det R| >= 2^-16 ||R||_F^3.  A rotation gives 3^-1.5; a (nearly) singular R would map
// some unit direction of Eq. 3 to (nearly) zero, a "ray" that has no exit face in the walk.
bool r360_poses_ok(const float* poses, int B) {
  if (!poses || B < 1) return false;
  for (int b = 0; b < B; ++b) {
    const float* P = poses + (size_t)b * 12;
    double r[9], sq = 0.0;
    for (int i = 0; i < 12; ++i)
      if (!std::isfinite(P[i])) return false;
    for (int row = 0; row < 3; ++row)
      for (int col = 0; col < 3; ++col) {
        const double v = (double)P[row * 4 + col];
        r[row * 3 + col] = v;
        sq += v * v;
      }
    const double nf = std::sqrt(sq);
    if (!(nf >= 0x1p-16 && nf <= 0x1p16)) return false;
    // det by the rule of Sarrus
    const double det = r[0] * r[4] * r[8] + r[1] * r[5] * r[6] + r[2] * r[3] * r[7] - r[2] * r[4] * r[6] -
                       r[1] * r[3] * r[8] - r[0] * r[5] * r[7];
    if (!(std::fabs(det) >= 0x1p-16 * nf * nf * nf)) return false;
  }
  return true;
}

r360_status r360_cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
  cudaGetLastError();  // clear the non-sticky error state
  return e == cudaErrorMemoryAllocation ? R360_ERR_OOM : R360_ERR_CUDA;
}

namespace r360 {
// defined in mlp_tc.cu: bf16 operand packing for the tensor-core kernel
size_t tc_pack_stride(const NetShape& net);
bool tc_pack_subfield(const NetShape& net, const float* src_blob, void* dst, int operand_f16);
size_t tc_smem_bytes(const NetShape& net);
}  // namespace r360

// Octant skip distances of the empty voxels (common.cuh): for the octant with direction signs (sx, sy, sz),
//   D(v) = 0 if v is occupied, else min(255, 1 + min over the 7 neighbours v + (ex sx, ey sy, ez sz), e in {0,1}^3 \ 0,
//   of D(neighbour)), a neighbour outside the grid counting as 255
// -- the cube of D voxels per axis that starts at v and extends in the octant's direction is empty iff v is empty
// and the seven cubes of D-1 voxels that start at those neighbours are.  One sweep per octant, against the
// direction of travel, so that every neighbour is final when it is read; the eight sweeps run on eight threads.
static bool skip_distances(const std::vector<uint16_t>& grid, const int dims[3], std::vector<uint8_t>& skip) {
  const int Nx = dims[0], Ny = dims[1], Nz = dims[2];
  const size_t N = (size_t)Nx * Ny * Nz;
  try { skip.assign(N * 8, 0); } catch (const std::bad_alloc&) { return false; }
  auto sweep = [&](int o) {
    const int sx = (o & 1) ? -1 : 1, sy = (o & 2) ? -1 : 1, sz = (o & 4) ? -1 : 1;
    auto at = [&](int x, int y, int z) -> int {
      if (x < 0 || x >= Nx || y < 0 || y >= Ny || z < 0 || z >= Nz) return 255;
      return skip[(((size_t)z * Ny + y) * Nx + x) * 8 + o];
    };
    for (int kz = 0; kz < Nz; ++kz) {
      const int z = sz > 0 ? Nz - 1 - kz : kz;
      for (int ky = 0; ky < Ny; ++ky) {
        const int y = sy > 0 ? Ny - 1 - ky : ky;
        for (int kx = 0; kx < Nx; ++kx) {
          const int x = sx > 0 ? Nx - 1 - kx : kx;
          const size_t v = ((size_t)z * Ny + y) * Nx + x;
          if (grid[v] < kEmptyBase) { skip[v * 8 + o] = 0; continue; }
          int m = 255;
          for (int e = 1; e < 8; ++e) {
            const int nb = at(x + ((e & 1) ? sx : 0), y + ((e & 2) ? sy : 0), z + ((e & 4) ? sz : 0));
            if (nb < m) m = nb;
          }
          skip[v * 8 + o] = (uint8_t)(m >= 254 ? 255 : m + 1);
        }
      }
    }
  };
  // the eight sweeps write disjoint bytes; whatever could not get a thread runs here
  std::thread th[8];
  int started = 0;
  try {
    for (; started < 7; ++started) th[started] = std::thread(sweep, started);
  } catch (...) {
  }
  for (int o = started; o < 8; ++o) sweep(o);
  for (int o = 0; o < started; ++o) th[o].join();
  return true;
}

extern "C" {

const char* r360_status_string(r360_status s) {
  switch (s) {
    case R360_OK: return "ok";
    case R360_ERR_INVALID_ARG: return "invalid argument";
    case R360_ERR_BAD_LABEL: return "occupied voxel with a subfield label outside [0, n)";
    case R360_ERR_NONFINITE: return "non-finite weight";
    case R360_ERR_CUDA: return "CUDA error";
    case R360_ERR_OOM: return "out of memory";
    case R360_ERR_CAPACITY: return "caller buffer too small";
  }
  return "unknown status";
}

const char* r360_last_cuda_error(void) { return g_cuda_err; }
const char* r360_version(void) { return "r360 0.1 sm_100a"; }

int64_t r360_params_per_subfield(const r360_scene_desc* desc) {
  if (!desc_ok(desc)) return 0;
  SrcLayout s;
  Fp32Layout t;
  make_layouts(*desc, s, t);
  return s.total;
}

void r360_scene_destroy(r360_scene* sc) {
  if (!sc) return;
  cudaFree(sc->d_grid); cudaFree(sc->d_skip); cudaFree(sc->d_frames); cudaFree(sc->d_wt); cudaFree(sc->d_wpack); cudaFree(sc->d_wpack_f16);
  cudaFree(sc->d_tables); cudaFree(sc->d_poses);
  cudaFree(sc->buf.ray_cnt); cudaFree(sc->buf.ray_off); cudaFree(sc->buf.block_sum);
  cudaFree(sc->buf.totals);     // one allocation: totals | bin_cnt | bin_ovf
  cudaFree(sc->buf.bin_start); cudaFree(sc->buf.bin_cursor);
  cudaFree(sc->buf.tile_start);
  cudaDeviceSynchronize();   // (work of the last calls may still use the buffers)
  cudaFree(sc->buf.seg_td); cudaFree(sc->buf.recs); cudaFree(sc->buf.out);
  cudaFree(sc->d_dirblk);
  cudaFree(sc->buf.hit_t); cudaFree(sc->buf.hit_lab);
  cudaFree(sc->buf.blk_list); cudaFree(sc->buf.blk_list_n);
  cudaFree(sc->d_pass_cnt); cudaFree(sc->buf.pass_off); cudaFree(sc->buf.st_c); cudaFree(sc->buf.st_T);
  for (int i = 0; i < 2; ++i) {
    cudaFree(sc->d_stage_rgb[i]); cudaFree(sc->d_stage_depth[i]);
    if (sc->ev_copy_done[i]) cudaEventDestroy(sc->ev_copy_done[i]);
  }
  if (sc->h_snap) cudaFreeHost(sc->h_snap);
  if (sc->h_poses) cudaFreeHost(sc->h_poses);
  if (sc->copy_stream) cudaStreamDestroy(sc->copy_stream);
  if (sc->ev_chunk_done) cudaEventDestroy(sc->ev_chunk_done);
  for (auto& ce : sc->events) {
    for (auto& e : ce.e) cudaEventDestroy(e);
    cudaEventDestroy(ce.scanned);
    cudaEventDestroy(ce.finished);
  }
  cudaGetLastError();
  delete sc;
}

r360_status r360_scene_create(const r360_scene_desc* desc, const uint8_t* occupancy,
                              const int32_t* voxel_subfield, const float* weights, r360_scene** out) {
  if (out) *out = nullptr;
  if (!out || !occupancy || !voxel_subfield || !weights || !desc_ok(desc)) return R360_ERR_INVALID_ARG;
  r360_scene* sc = new (std::nothrow) r360_scene();
  if (!sc) return R360_ERR_OOM;
  struct Guard {
    r360_scene* s;
    ~Guard() { if (s) r360_scene_destroy(s); }
  } guard{sc};
  sc->desc = *desc;
  const int n = desc->n_subfields, Wd = desc->hidden_width;
  const long long N = (long long)desc->dims[0] * desc->dims[1] * desc->dims[2];
  // geometry (reading C): voxel size = (box_max - box_min) / dims, one subtract, one divide
  GridParams& g = sc->grid_p;
  for (int a = 0; a < 3; ++a) {
    g.dims[a] = desc->dims[a];
    g.box_min[a] = desc->box_min[a];
    volatile float ext = desc->box_max[a] - desc->box_min[a];
    g.vs[a] = ext / (float)desc->dims[a];
    g.inv_vs[a] = 1.0f / g.vs[a];
  }
  g.K = desc->samples_per_voxel;
  g.Kf = (float)g.K;
  g.Kinv = (g.K > 0 && (g.K & (g.K - 1)) == 0) ? 1.0f / (float)g.K : 0.0f;
  sc->segs_per_tile = kTileRows / g.K;
  NetShape& net = sc->net;
  net.Wd = Wd; net.Hd = desc->n_hidden; net.Lp = desc->pe_pos_levels; net.Ld = desc->pe_dir_levels;
  net.pe_p = pe_dim(net.Lp); net.pe_d = pe_dim(net.Ld); net.act = desc->density_activation;
  SrcLayout src;
  make_layouts(*desc, src, sc->lay);
  net.P = src.total;

  // fused grid + per-subfield voxel bounding boxes (reading A3)
  std::vector<uint16_t> grid;
  std::vector<int> lo, hi;
  try {
    grid.resize((size_t)N);
    lo.assign((size_t)n * 3, std::numeric_limits<int>::max());
    hi.assign((size_t)n * 3, -1);
  } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
  for (long long v = 0; v < N; ++v) {
    if (occupancy[v] < desc->occ_threshold) { grid[(size_t)v] = (uint16_t)0xFFFFu; continue; }
    int k = voxel_subfield[v];
    if (k < 0 || k >= n) return R360_ERR_BAD_LABEL;
    grid[(size_t)v] = (uint16_t)k;
    int idx[3] = {(int)(v % g.dims[0]), (int)((v / g.dims[0]) % g.dims[1]),
                  (int)(v / ((long long)g.dims[0] * g.dims[1]))};
    for (int a = 0; a < 3; ++a) {
      if (idx[a] < lo[(size_t)k * 3 + a]) lo[(size_t)k * 3 + a] = idx[a];
      if (idx[a] > hi[(size_t)k * 3 + a]) hi[(size_t)k * 3 + a] = idx[a];
    }
  }
  std::vector<uint8_t> skip;
  if (!skip_distances(grid, g.dims, skip)) return R360_ERR_OOM;
  for (long long i = 0; i < (long long)n * src.total; ++i)
    if (!std::isfinite(weights[i])) return R360_ERR_NONFINITE;
  std::vector<SubfieldFrame> frames;
  try { frames.resize((size_t)n); } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
  for (int k = 0; k < n; ++k) {
    float c[3], ih[3];
    for (int a = 0; a < 3; ++a) {
      if (hi[(size_t)k * 3 + a] < 0) { c[a] = 0.0f; ih[a] = 1.0f; continue; }
      // planes from the index: box_min + k*s (one multiply, one add), then centre and half extent
      volatile float ml = (float)lo[(size_t)k * 3 + a] * g.vs[a];
      volatile float mh = (float)(hi[(size_t)k * 3 + a] + 1) * g.vs[a];
      volatile float pl = g.box_min[a] + ml;
      volatile float ph = g.box_min[a] + mh;
      volatile float sum = pl + ph;
      volatile float dif = ph - pl;
      volatile float h = 0.5f * dif;
      c[a] = 0.5f * sum;
      ih[a] = 1.0f / h;
    }
    frames[(size_t)k] = SubfieldFrame{c[0], c[1], c[2], 0.f, ih[0], ih[1], ih[2], 0.f};
  }
  // fp32 weights, transposed + padded
  const Fp32Layout& lay = sc->lay;
  std::vector<float> wt;
  try { wt.assign((size_t)n * lay.total, 0.0f); } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
  for (int k = 0; k < n; ++k) {
    const float* s = weights + (size_t)k * src.total;
    float* d = wt.data() + (size_t)k * lay.total;
    for (int l = 0; l < net.Hd; ++l)
      transpose_layer(s + src.trunk[l], d + lay.trunk[l], Wd, l == 0 ? net.pe_p : Wd, Wd);
    for (int i = 0; i <= Wd; ++i) d[lay.dens + i] = s[src.dens + i];     // w[Wd] then b
    transpose_layer(s + src.feat, d + lay.feat, Wd, Wd, Wd);
    transpose_layer(s + src.col, d + lay.col, Wd, Wd + net.pe_d, Wd);
    transpose_layer(s + src.rgb, d + lay.rgb, 3, Wd, 4);
  }
  // bf16 operand tiles for the tensor-core kernel
  sc->wpack_stride = tc_pack_stride(net);
  // (a network whose weight buffers do not fit the kernel's shared memory is refused at
  // r360_set_precision, not at render time)
  sc->tc_fits = sc->wpack_stride && tc_smem_bytes(net) <= 227 * 1024;
  if (!sc->tc_fits) sc->wpack_stride = 0;
  std::vector<unsigned char> wpack, wpack16;
  bool f16_ok = true;
  if (sc->wpack_stride) {
    try {
      wpack.assign((size_t)n * sc->wpack_stride, 0);
      wpack16.assign((size_t)n * sc->wpack_stride, 0);
    } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
    for (int k = 0; k < n; ++k) {
      tc_pack_subfield(net, weights + (size_t)k * src.total, wpack.data() + (size_t)k * sc->wpack_stride, 0);
      f16_ok = tc_pack_subfield(net, weights + (size_t)k * src.total, wpack16.data() + (size_t)k * sc->wpack_stride, 1) && f16_ok;
    }
  }

  int dev = 0;
  R360_CUDA(cudaGetDevice(&dev));
  R360_CUDA(cudaDeviceGetAttribute(&sc->n_sms, cudaDevAttrMultiProcessorCount, dev));
  R360_CUDA(cudaMalloc(&sc->d_grid, (size_t)N * sizeof(uint16_t)));
  R360_CUDA(cudaMalloc(&sc->d_frames, (size_t)n * sizeof(SubfieldFrame)));
  R360_CUDA(cudaMalloc(&sc->d_wt, wt.size() * sizeof(float)));
  R360_CUDA(cudaMemcpy(sc->d_grid, grid.data(), (size_t)N * sizeof(uint16_t), cudaMemcpyHostToDevice));
  R360_CUDA(cudaMalloc(&sc->d_skip, skip.size()));
  R360_CUDA(cudaMemcpy(sc->d_skip, skip.data(), skip.size(), cudaMemcpyHostToDevice));
  sc->grid_p.skip = sc->d_skip;
  R360_CUDA(cudaMemcpy(sc->d_frames, frames.data(), (size_t)n * sizeof(SubfieldFrame), cudaMemcpyHostToDevice));
  R360_CUDA(cudaMemcpy(sc->d_wt, wt.data(), wt.size() * sizeof(float), cudaMemcpyHostToDevice));
  if (!wpack.empty()) {
    R360_CUDA(cudaMalloc(&sc->d_wpack, wpack.size()));
    R360_CUDA(cudaMemcpy(sc->d_wpack, wpack.data(), wpack.size(), cudaMemcpyHostToDevice));
    if (f16_ok) {
      R360_CUDA(cudaMalloc(&sc->d_wpack_f16, wpack16.size()));
      R360_CUDA(cudaMemcpy(sc->d_wpack_f16, wpack16.data(), wpack16.size(), cudaMemcpyHostToDevice));
    }
  }
  // the counters that are cleared at the start of a chunk sit in ONE allocation, cleared by one memset:
  // totals[kTotN] | bin_cnt[n] | bin_ovf[n]
  R360_CUDA(cudaMalloc(&sc->buf.totals, kTotN * sizeof(unsigned long long) + (size_t)n * 8));
  sc->buf.bin_cnt = reinterpret_cast<uint32_t*>(sc->buf.totals + kTotN);
  sc->buf.bin_ovf = sc->buf.bin_cnt + n;
  R360_CUDA(cudaMalloc(&sc->buf.bin_start, (size_t)(n + 1) * 4));
  R360_CUDA(cudaMalloc(&sc->buf.bin_cursor, (size_t)n * 4));
  R360_CUDA(cudaMalloc(&sc->buf.tile_start, (size_t)(n + 1) * 4));
  {
    const size_t bytes = (size_t)r360_scene::kMaxChunks * 2 * kTotN * sizeof(unsigned long long);
    R360_CUDA(cudaHostAlloc(&sc->h_snap, bytes, cudaHostAllocMapped));
    std::memset(sc->h_snap, 0, bytes);
    R360_CUDA(cudaHostGetDevicePointer(&sc->d_snap, sc->h_snap, 0));
  }
  guard.s = nullptr;
  *out = sc;
  return R360_OK;
}

}  // extern "C"
