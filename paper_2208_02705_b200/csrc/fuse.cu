// r360 -- progressive probabilistic occupancy (Eq. 6; Algorithm 1 stage I :139-146): one
// observation = a depth panorama (Eq. 4), optionally with an uncertainty panorama, fused into the log-odds grid
//     logit(p | z_1:t) = logit(p | z_1:t-1) + logit(p | z_t),  logit in [-2, 3.5]  (:119-122).
// Readings O1-O5: natural-log odds clamped after every observation; Octomap's scan insertion (the
// framework the paper adopts, :128): per observation a voxel is updated once, "occupied" if a ray ends in it, else
// "free" if a ray crosses it before its end; l_free = ln(0.4/0.6), l_occ = ln(p/(1-p)), p = 0.5 + 0.2 (1 - u) with
// u the smallest uncertainty of the rays ending in the voxel (Octomap's defaults 0.7 / 0.4 for u = 0; its default
// clamps are the paper's -2 / 3.5); rays and the walk are readings B and C of the renderer.
//   k_mark   : one thread per pixel walks every voxel its ray crosses up to the end point and sets a flag
//              (atomicOr: free / occupied) and, for the end-point voxel, the minimum uncertainty (atomicMin on
//              the bits of a non-negative float)
//   k_update : one thread per voxel applies Eq. 6 once and clears the flags
// The result does not depend on the order of the rays (flags and a minimum), so it is reproducible bit for bit.
#include <cmath>
#include <cstdio>
#include <mutex>
#include <new>
#include <vector>

#include "scene.h"

namespace {

using namespace r360;

constexpr uint32_t kFree = 1u, kOcc = 2u;

// plain voxel walk of reading C (every crossed voxel, no skipping): the renderer's Walker returns occupied voxels
// only and needs the skip grid; here the grid is what is being estimated
__global__ void __launch_bounds__(256)
k_mark(GridParams g, FrameParams f, const float* __restrict__ depth, const float* __restrict__ unc,
       uint32_t* __restrict__ flags, uint32_t* __restrict__ umin) {
  const unsigned r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= f.n_rays) return;
  const float D = depth[r];
  if (!(D > 0.0f) || !isfinite(D)) return;                      // O4
  const Ray ray = make_ray(f, r);
  float o[3], inv[3];
  bool par[3], neg[3];
  bool alive = true;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    o[a] = ray.o[a];
    par[a] = fabsf(ray.d[a]) < kParallelEps;
    neg[a] = ray.d[a] < 0.0f;
    inv[a] = par[a] ? 0.0f : __fdiv_rn(1.0f, ray.d[a]);
  }
  auto t_at = [&](int a, int k) { return __fmul_rn(__fsub_rn(plane(g, a, k), o[a]), inv[a]); };
  float t0 = 0.0f, t1 = __int_as_float(0x7f800000);
#pragma unroll
  for (int a = 0; a < 3; ++a) {                                 // C2
    const int N = g.dims[a];
    if (par[a]) {
      if (!(o[a] >= g.box_min[a] && o[a] < plane(g, a, N))) alive = false;
    } else {
      const float n_ = t_at(a, neg[a] ? N : 0), f_ = t_at(a, neg[a] ? 0 : N);
      if (n_ > t0) t0 = n_;
      if (f_ < t1) t1 = f_;
    }
  }
  if (!(t0 < t1)) alive = false;
  int idx[3];
  float tn[3], tf[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {                                 // C3
    const float pa = __fmaf_rn(t0, ray.d[a], o[a]);
    const float fl = floorf(__fdiv_rn(__fsub_rn(pa, g.box_min[a]), g.vs[a]));
    const int N = g.dims[a];
    idx[a] = (fl < 0.0f) ? 0 : ((fl > (float)(N - 1)) ? N - 1 : (int)fl);
    tn[a] = par[a] ? __int_as_float(0xff800000) : t_at(a, idx[a] + (neg[a] ? 1 : 0));
    tf[a] = par[a] ? __int_as_float(0x7f800000) : t_at(a, idx[a] + (neg[a] ? 0 : 1));
  }
  const float u = unc ? fminf(fmaxf(unc[r], 0.0f), 1.0f) : 0.0f;
  while (alive) {                                               // C4
    const float ti = fmaxf(fmaxf(t0, tn[0]), fmaxf(tn[1], tn[2]));
    int amin = 2;
    float to = tf[2];
    if (tf[1] <= to) { to = tf[1]; amin = 1; }
    if (tf[0] <= to) { to = tf[0]; amin = 0; }
    if (ti < to) {                                              // crossed
      if (!(ti < D)) break;                                     // the ray ended before this voxel
      const size_t v = ((size_t)idx[2] * g.dims[1] + idx[1]) * g.dims[0] + idx[0];
      if (D < to) {                                             // the end point lies in this voxel
        atomicOr(&flags[v], kOcc);
        atomicMin(&umin[v], __float_as_uint(u));                // u >= 0: the bit patterns order like the values
        break;
      }
      atomicOr(&flags[v], kFree);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (a == amin) {
        idx[a] += neg[a] ? -1 : 1;
        tn[a] = tf[a];
        tf[a] = t_at(a, idx[a] + (neg[a] ? 0 : 1));
        if (idx[a] < 0 || idx[a] >= g.dims[a]) alive = false;
      }
    }
  }
}

__global__ void __launch_bounds__(256)
k_update(size_t N, float l_free, float* __restrict__ L, uint32_t* __restrict__ flags, uint32_t* __restrict__ umin) {
  const size_t v = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= N) return;
  const uint32_t fl = flags[v];
  if (!fl) return;
  float inc = l_free;
  if (fl & kOcc) {
    // O3: p = 0.5 + 0.2 (1 - u) in binary32; l = ln(p / (1 - p)) in binary64, rounded once
    const float u = __uint_as_float(umin[v]);
    const float p = __fadd_rn(0.5f, __fmul_rn(0.2f, __fsub_rn(1.0f, u)));
    inc = (float)log((double)p / (1.0 - (double)p));
  }
  L[v] = fminf(3.5f, fmaxf(-2.0f, __fadd_rn(L[v], inc)));       // O1
  flags[v] = 0;
  umin[v] = 0x3F800000u;
}

__global__ void __launch_bounds__(256) k_fill_u32(uint32_t* __restrict__ p, size_t n, uint32_t v) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// voxel occupied iff logit > ln(0.97 / 0.03) (reading O5): the uint8 occupancy of r360_scene_create
__global__ void __launch_bounds__(256) k_threshold(const float* __restrict__ L, size_t n, float thr, uint8_t* __restrict__ occ) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) occ[i] = L[i] > thr ? 255 : 0;
}

}  // namespace

// The log-odds grid stays on the device between observations (Algorithm 1 stage I fuses T panoramas
// progressively): no per-observation allocation, no grid crossing PCIe.
struct r360_fusion {
  r360::GridParams g{};
  size_t N = 0;
  float* d_L = nullptr;
  uint32_t* d_flags = nullptr;        // kFree | kOcc of the observation being fused; zero between observations
  uint32_t* d_umin = nullptr;         // bits of the smallest uncertainty per voxel; 1.0f between observations
  float* d_tab = nullptr;             // trig tables of the last image size
  int tab_W = 0, tab_H = 0;
  float* d_pose = nullptr;
  float* d_depth = nullptr;           // staging of host images
  float* d_unc = nullptr;
  size_t img_cap = 0;
  uint8_t* d_occ = nullptr;           // r360_fusion_read: thresholded grid
};

extern "C" {

void r360_fusion_destroy(r360_fusion* fu) {
  if (!fu) return;
  cudaFree(fu->d_L); cudaFree(fu->d_flags); cudaFree(fu->d_umin); cudaFree(fu->d_tab); cudaFree(fu->d_pose);
  cudaFree(fu->d_depth); cudaFree(fu->d_unc); cudaFree(fu->d_occ);
  cudaGetLastError();
  delete fu;
}

r360_status r360_fusion_create(const int32_t dims[3], const float box_min[3], const float box_max[3],
                               const float* logodds_init, r360_fusion** out) {
  if (out) *out = nullptr;
  if (!dims || !box_min || !box_max || !out) return R360_ERR_INVALID_ARG;
  r360_fusion* fu = new (std::nothrow) r360_fusion();
  if (!fu) return R360_ERR_OOM;
  struct Guard {
    r360_fusion* f;
    ~Guard() { if (f) r360_fusion_destroy(f); }
  } guard{fu};
  for (int a = 0; a < 3; ++a) {
    if (dims[a] < 1 || !(box_max[a] > box_min[a])) return R360_ERR_INVALID_ARG;
    fu->g.dims[a] = dims[a];
    fu->g.box_min[a] = box_min[a];
    volatile float ext = box_max[a] - box_min[a];               // voxel size exactly as the renderer computes it
    fu->g.vs[a] = ext / (float)dims[a];
    fu->g.inv_vs[a] = 1.0f / fu->g.vs[a];
  }
  if ((long long)dims[0] * dims[1] * dims[2] > (1ll << 31) - 1) return R360_ERR_INVALID_ARG;
  const size_t N = fu->N = (size_t)dims[0] * dims[1] * dims[2];
  R360_CUDA(cudaMalloc(&fu->d_L, N * sizeof(float)));
  R360_CUDA(cudaMalloc(&fu->d_flags, N * sizeof(uint32_t)));
  R360_CUDA(cudaMalloc(&fu->d_umin, N * sizeof(uint32_t)));
  R360_CUDA(cudaMalloc(&fu->d_pose, 12 * sizeof(float)));
  if (logodds_init) R360_CUDA(cudaMemcpy(fu->d_L, logodds_init, N * sizeof(float), cudaMemcpyHostToDevice));
  else R360_CUDA(cudaMemset(fu->d_L, 0, N * sizeof(float)));
  R360_CUDA(cudaMemset(fu->d_flags, 0, N * sizeof(uint32_t)));
  k_fill_u32<<<(unsigned)((N + 255) / 256), 256>>>(fu->d_umin, N, 0x3F800000u);   // umin starts at 1.0
  R360_CUDA(cudaGetLastError());
  R360_CUDA(cudaDeviceSynchronize());
  guard.f = nullptr;
  *out = fu;
  return R360_OK;
}

// depth / uncertainty: DEVICE pointers (for example the depth output of r360_render)
r360_status r360_fusion_fuse_device(r360_fusion* fu, const float pose[12], int32_t W, int32_t H, const float* depth,
                                    const float* uncertainty) {
  if (!fu || !pose || !depth || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if ((long long)W * H >= (1ll << 30)) return R360_ERR_INVALID_ARG;
  if (!r360_poses_ok(pose, 1)) return R360_ERR_INVALID_ARG;     // non-finite or (nearly) singular (reading B5)
  if (!fu->d_tab || fu->tab_W != W || fu->tab_H != H) {
    // reading B2: trig of the pixel-centre angles in binary64, rounded once
    const double kPi = 3.14159265358979323846;
    std::vector<float> tab;
    try { tab.resize((size_t)2 * W + 2 * H); } catch (const std::bad_alloc&) { return R360_ERR_OOM; }
    for (int i = 0; i < W; ++i) {
      const double phi = (((double)i + 0.5) - (double)W / 2.0) * (2.0 * kPi / (double)W);
      tab[i] = (float)std::sin(phi);
      tab[(size_t)W + i] = (float)std::cos(phi);
    }
    for (int j = 0; j < H; ++j) {
      const double theta = -((((double)j + 0.5) - (double)H / 2.0) * (kPi / (double)H));
      tab[(size_t)2 * W + j] = (float)std::sin(theta);
      tab[(size_t)2 * W + H + j] = (float)std::cos(theta);
    }
    cudaFree(fu->d_tab);
    fu->d_tab = nullptr;
    R360_CUDA(cudaMalloc(&fu->d_tab, tab.size() * sizeof(float)));
    R360_CUDA(cudaMemcpy(fu->d_tab, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice));
    fu->tab_W = W;
    fu->tab_H = H;
  }
  R360_CUDA(cudaMemcpy(fu->d_pose, pose, 12 * sizeof(float), cudaMemcpyHostToDevice));
  const size_t R = (size_t)W * H;
  r360::FrameParams f{};
  f.W = W; f.H = H; f.ray0 = 0; f.pose0 = 0; f.pix0 = 0; f.n_rays = (unsigned)R; f.camera = 0;
  f.poses = fu->d_pose;
  f.sin_phi = fu->d_tab; f.cos_phi = fu->d_tab + W;
  f.sin_theta = fu->d_tab + 2 * (size_t)W; f.cos_theta = fu->d_tab + 2 * (size_t)W + H;
  k_mark<<<(unsigned)((R + 255) / 256), 256>>>(fu->g, f, depth, uncertainty, fu->d_flags, fu->d_umin);
  k_update<<<(unsigned)((fu->N + 255) / 256), 256>>>(fu->N, (float)std::log(0.4 / 0.6), fu->d_L, fu->d_flags, fu->d_umin);
  R360_CUDA(cudaGetLastError());
  return R360_OK;
}

// depth / uncertainty: HOST pointers
r360_status r360_fusion_fuse(r360_fusion* fu, const float pose[12], int32_t W, int32_t H, const float* depth,
                             const float* uncertainty) {
  if (!fu || !pose || !depth || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if ((long long)W * H >= (1ll << 30)) return R360_ERR_INVALID_ARG;
  const size_t R = (size_t)W * H;
  if (R > fu->img_cap) {
    cudaFree(fu->d_depth); cudaFree(fu->d_unc);
    fu->d_depth = fu->d_unc = nullptr;
    fu->img_cap = 0;
    R360_CUDA(cudaMalloc(&fu->d_depth, R * sizeof(float)));
    R360_CUDA(cudaMalloc(&fu->d_unc, R * sizeof(float)));
    fu->img_cap = R;
  }
  R360_CUDA(cudaMemcpy(fu->d_depth, depth, R * sizeof(float), cudaMemcpyHostToDevice));
  if (uncertainty) R360_CUDA(cudaMemcpy(fu->d_unc, uncertainty, R * sizeof(float), cudaMemcpyHostToDevice));
  return r360_fusion_fuse_device(fu, pose, W, H, fu->d_depth, uncertainty ? fu->d_unc : nullptr);
}

r360_status r360_fusion_read(r360_fusion* fu, float* logodds_out, uint8_t* occupancy_out) {
  if (!fu || (!logodds_out && !occupancy_out)) return R360_ERR_INVALID_ARG;
  if (logodds_out) R360_CUDA(cudaMemcpy(logodds_out, fu->d_L, fu->N * sizeof(float), cudaMemcpyDeviceToHost));
  if (occupancy_out) {
    if (!fu->d_occ) R360_CUDA(cudaMalloc(&fu->d_occ, fu->N));
    k_threshold<<<(unsigned)((fu->N + 255) / 256), 256>>>(fu->d_L, fu->N, (float)std::log(0.97 / 0.03), fu->d_occ);
    R360_CUDA(cudaGetLastError());
    R360_CUDA(cudaMemcpy(occupancy_out, fu->d_occ, fu->N, cudaMemcpyDeviceToHost));
  }
  return R360_OK;
}

// one observation on a host grid: create, fuse, read, destroy
r360_status r360_occupancy_fuse(const int32_t dims[3], const float box_min[3], const float box_max[3],
                                float* logodds, const float pose[12], int32_t W, int32_t H,
                                const float* depth, const float* uncertainty) {
  if (!dims || !box_min || !box_max || !logodds || !pose || !depth || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  r360_fusion* fu = nullptr;
  r360_status st = r360_fusion_create(dims, box_min, box_max, logodds, &fu);
  if (st != R360_OK) return st;
  st = r360_fusion_fuse(fu, pose, W, H, depth, uncertainty);
  if (st == R360_OK) st = r360_fusion_read(fu, logodds, nullptr);
  r360_fusion_destroy(fu);
  return st;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// r360_fusion_fuse_static: one observation of Eq. 6 for callers that must not allocate device memory.
//
// Who that is: a host program that has handed the whole GPU to its own arena or caching allocator (a later
// cudaMalloc from a library would fail or fragment it), a frame loop that cannot take the device-wide stall a
// cudaMalloc / cudaFree may cause, and code that runs while allocation is forbidden in its process (for example
// while some other thread records a CUDA graph in the global capture mode).  The r360_fusion handle allocates at
// create time and again whenever the image size changes; this entry point never allocates: the per-voxel flags, the
// per-voxel minimum uncertainty, the pixel-angle tables and the pose live in ONE file-scope device array of fixed
// size.  The price is a fixed limit (R360_STATIC_MAX_VOXELS, R360_STATIC_MAX_W, R360_STATIC_MAX_H) and
// kStaticBytes (64 MiB + 48 KiB) of device memory on every GPU that loads libr360.so, from load until exit.
//
// In host code the name g_fuse_scratch is only a handle for the runtime, not a device address: the address comes
// from cudaGetSymbolAddress, asked once per device with that device current (static_scratch below).
namespace {

constexpr size_t kStaticMaxVoxels = R360_STATIC_MAX_VOXELS;
constexpr int kStaticMaxW = R360_STATIC_MAX_W, kStaticMaxH = R360_STATIC_MAX_H;
constexpr size_t kStaticTabFloats = 2 * (size_t)kStaticMaxW + 2 * (size_t)kStaticMaxH;
// layout: flags uint32[kStaticMaxVoxels] | umin uint32[kStaticMaxVoxels] | tables float[kStaticTabFloats] | pose float[16]
constexpr size_t kStaticOffUmin = kStaticMaxVoxels * sizeof(uint32_t);
constexpr size_t kStaticOffTab = 2 * kStaticOffUmin;
constexpr size_t kStaticOffPose = kStaticOffTab + kStaticTabFloats * sizeof(float);
constexpr size_t kStaticBytes = kStaticOffPose + 16 * sizeof(float);
static_assert(kStaticOffTab % 256 == 0 && kStaticOffPose % 256 == 0, "sub-buffers keep the array's alignment");

static __device__ __align__(256) unsigned char g_fuse_scratch[kStaticBytes];

constexpr int kStaticMaxDevices = 64;
struct StaticDev {
  unsigned char* base = nullptr;    // device address of g_fuse_scratch on this device
  int tab_W = 0, tab_H = 0;         // image size the tables in the scratch were built for
};
StaticDev g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;

// set-up, once per device, with that device current
r360_status static_scratch(StaticDev** out) {
  int dev = -1;
  R360_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return R360_ERR_INVALID_ARG;
  StaticDev& sd = g_static_dev[dev];
  if (!sd.base) {
    void* p = nullptr;
    R360_CUDA(cudaGetSymbolAddress(&p, g_fuse_scratch));
    if (!p) return R360_ERR_CUDA;
    sd.base = static_cast<unsigned char*>(p);
  }
  *out = &sd;
  return R360_OK;
}

}  // namespace

extern "C" r360_status r360_fusion_fuse_static(const int32_t dims[3], const float box_min[3], const float box_max[3],
                                               float* logodds, const float pose[12], int32_t W, int32_t H,
                                               const float* depth, const float* uncertainty, void* cuda_stream) {
  if (!dims || !box_min || !box_max || !logodds || !pose || !depth || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  r360::GridParams g{};
  for (int a = 0; a < 3; ++a) {
    if (dims[a] < 1 || !(box_max[a] > box_min[a])) return R360_ERR_INVALID_ARG;
    g.dims[a] = dims[a];
    g.box_min[a] = box_min[a];
    volatile float ext = box_max[a] - box_min[a];               // voxel size exactly as r360_fusion_create computes it
    g.vs[a] = ext / (float)dims[a];
    g.inv_vs[a] = 1.0f / g.vs[a];
  }
  if (!r360_poses_ok(pose, 1)) return R360_ERR_INVALID_ARG;     // non-finite or (nearly) singular (reading B5)
  const unsigned long long N64 = (unsigned long long)dims[0] * (unsigned long long)dims[1] * (unsigned long long)dims[2];
  if (N64 > kStaticMaxVoxels || W > kStaticMaxW || H > kStaticMaxH) {
    // the text r360_last_cuda_error() returns names the limit that was hit
    char msg[200];
    snprintf(msg, sizeof(msg), "r360_fusion_fuse_static: %llu voxels, %d x %d image exceed the static scratch "
             "(at most %zu voxels, %d x %d)", N64, W, H, kStaticMaxVoxels, kStaticMaxW, kStaticMaxH);
    r360_cuda_fail(cudaErrorInvalidValue, msg);
    return R360_ERR_CAPACITY;
  }
  const size_t N = (size_t)N64, R = (size_t)W * H;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  std::lock_guard<std::mutex> lock(g_static_mu);
  StaticDev* sd = nullptr;
  const r360_status st = static_scratch(&sd);
  if (st != R360_OK) return st;
  uint32_t* flags = reinterpret_cast<uint32_t*>(sd->base);
  uint32_t* umin = reinterpret_cast<uint32_t*>(sd->base + kStaticOffUmin);
  float* d_tab = reinterpret_cast<float*>(sd->base + kStaticOffTab);
  float* d_pose = reinterpret_cast<float*>(sd->base + kStaticOffPose);
  if (sd->tab_W != W || sd->tab_H != H) {
    // reading B2: trig of the pixel-centre angles in binary64, rounded once (the same expressions as above).  The
    // source is pageable stack memory: cudaMemcpyAsync has staged it when it returns.
    const double kPi = 3.14159265358979323846;
    float tab[kStaticTabFloats];
    for (int i = 0; i < W; ++i) {
      const double phi = (((double)i + 0.5) - (double)W / 2.0) * (2.0 * kPi / (double)W);
      tab[i] = (float)std::sin(phi);
      tab[(size_t)W + i] = (float)std::cos(phi);
    }
    for (int j = 0; j < H; ++j) {
      const double theta = -((((double)j + 0.5) - (double)H / 2.0) * (kPi / (double)H));
      tab[(size_t)2 * W + j] = (float)std::sin(theta);
      tab[(size_t)2 * W + H + j] = (float)std::cos(theta);
    }
    sd->tab_W = sd->tab_H = 0;
    R360_CUDA(cudaMemcpyAsync(d_tab, tab, ((size_t)2 * W + 2 * H) * sizeof(float), cudaMemcpyHostToDevice, stream));
    sd->tab_W = W;
    sd->tab_H = H;
  }
  R360_CUDA(cudaMemcpyAsync(d_pose, pose, 12 * sizeof(float), cudaMemcpyHostToDevice, stream));
  // the array keeps what the last call (any grid size, possibly a failed one) left in it: the part this call uses
  // starts from "no flag, uncertainty 1.0" again
  R360_CUDA(cudaMemsetAsync(flags, 0, N * sizeof(uint32_t), stream));
  k_fill_u32<<<(unsigned)((N + 255) / 256), 256, 0, stream>>>(umin, N, 0x3F800000u);
  r360::FrameParams f{};
  f.W = W; f.H = H; f.ray0 = 0; f.pose0 = 0; f.pix0 = 0; f.n_rays = (unsigned)R; f.camera = 0;
  f.poses = d_pose;
  f.sin_phi = d_tab; f.cos_phi = d_tab + W;
  f.sin_theta = d_tab + 2 * (size_t)W; f.cos_theta = d_tab + 2 * (size_t)W + H;
  k_mark<<<(unsigned)((R + 255) / 256), 256, 0, stream>>>(g, f, depth, uncertainty, flags, umin);
  k_update<<<(unsigned)((N + 255) / 256), 256, 0, stream>>>(N, (float)std::log(0.4 / 0.6), logodds, flags, umin);
  R360_CUDA(cudaGetLastError());
  return R360_OK;
}
