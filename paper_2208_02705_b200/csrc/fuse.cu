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

}  // namespace

extern "C" r360_status r360_occupancy_fuse(const int32_t dims[3], const float box_min[3], const float box_max[3],
                                           float* logodds, const float pose[12], int32_t W, int32_t H,
                                           const float* depth, const float* uncertainty) {
  if (!dims || !box_min || !box_max || !logodds || !pose || !depth || W < 1 || H < 1) return R360_ERR_INVALID_ARG;
  if ((long long)W * H >= (1ll << 30)) return R360_ERR_INVALID_ARG;
  GridParams g{};
  for (int a = 0; a < 3; ++a) {
    if (dims[a] < 1 || !(box_max[a] > box_min[a])) return R360_ERR_INVALID_ARG;
    g.dims[a] = dims[a];
    g.box_min[a] = box_min[a];
    volatile float ext = box_max[a] - box_min[a];               // voxel size exactly as the renderer computes it
    g.vs[a] = ext / (float)dims[a];
    g.inv_vs[a] = 1.0f / g.vs[a];
  }
  for (int i = 0; i < 12; ++i)
    if (!std::isfinite(pose[i])) return R360_ERR_INVALID_ARG;
  const size_t N = (size_t)dims[0] * dims[1] * dims[2], R = (size_t)W * H;
  // reading B2: trig of the pixel-centre angles in binary64, rounded once
  const double kPi = 3.14159265358979323846;
  std::vector<float> tab((size_t)2 * W + 2 * H);
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
  float *d_L = nullptr, *d_tab = nullptr, *d_pose = nullptr, *d_depth = nullptr, *d_unc = nullptr;
  uint32_t *d_flags = nullptr, *d_umin = nullptr;
  r360_status rc = R360_OK;
#define U_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { rc = r360_cuda_fail(e_, #call); goto done; } } while (0)
  {
    std::vector<uint32_t> ones(N, 0x3F800000u);                 // umin starts at 1.0
    FrameParams f{};
    U_CUDA(cudaMalloc(&d_L, N * sizeof(float)));
    U_CUDA(cudaMalloc(&d_flags, N * sizeof(uint32_t)));
    U_CUDA(cudaMalloc(&d_umin, N * sizeof(uint32_t)));
    U_CUDA(cudaMalloc(&d_tab, tab.size() * sizeof(float)));
    U_CUDA(cudaMalloc(&d_pose, 12 * sizeof(float)));
    U_CUDA(cudaMalloc(&d_depth, R * sizeof(float)));
    if (uncertainty) U_CUDA(cudaMalloc(&d_unc, R * sizeof(float)));
    U_CUDA(cudaMemcpy(d_L, logodds, N * sizeof(float), cudaMemcpyHostToDevice));
    U_CUDA(cudaMemset(d_flags, 0, N * sizeof(uint32_t)));
    U_CUDA(cudaMemcpy(d_umin, ones.data(), N * sizeof(uint32_t), cudaMemcpyHostToDevice));
    U_CUDA(cudaMemcpy(d_tab, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice));
    U_CUDA(cudaMemcpy(d_pose, pose, 12 * sizeof(float), cudaMemcpyHostToDevice));
    U_CUDA(cudaMemcpy(d_depth, depth, R * sizeof(float), cudaMemcpyHostToDevice));
    if (uncertainty) U_CUDA(cudaMemcpy(d_unc, uncertainty, R * sizeof(float), cudaMemcpyHostToDevice));
    f.W = W; f.H = H; f.ray0 = 0; f.pose0 = 0; f.pix0 = 0; f.n_rays = (unsigned)R; f.camera = 0;
    f.poses = d_pose;
    f.sin_phi = d_tab; f.cos_phi = d_tab + W; f.sin_theta = d_tab + 2 * (size_t)W; f.cos_theta = d_tab + 2 * (size_t)W + H;
    k_mark<<<(unsigned)((R + 255) / 256), 256>>>(g, f, d_depth, d_unc, d_flags, d_umin);
    k_update<<<(unsigned)((N + 255) / 256), 256>>>(N, (float)std::log(0.4 / 0.6), d_L, d_flags, d_umin);
    U_CUDA(cudaGetLastError());
    U_CUDA(cudaMemcpy(logodds, d_L, N * sizeof(float), cudaMemcpyDeviceToHost));
  }
done:
#undef U_CUDA
  cudaFree(d_L); cudaFree(d_flags); cudaFree(d_umin); cudaFree(d_tab); cudaFree(d_pose); cudaFree(d_depth); cudaFree(d_unc);
  return rc;
}
