// r360 -- floorplan estimation from the occupancy map (section 5.0.2; Fig. 6):
//   project the occupied voxels of the upper slice (60-65 % of the height) to the floor plane, apply "simple
//   morphological operations", segment out the interior and its inner boundary, then add the occupied voxels of
//   the lower slice (20-30 %) that lie inside it.
// Readings F1-F7: height axis = grid z; a layer belongs to a slice iff its centre fraction lies in it;
// projection = OR over the layers; morphology = one closing by the 3x3 square (dilation with empty outside, erosion
// with set outside); interior = the 4-connected component of the non-wall cells that holds the seed cell; inner
// boundary = interior cells with a 4-neighbour that is not interior; obstacles = lower-slice cells in the interior.
// All images are Ny x Nx bytes on the device; the flood fill relaxes 32x32 tiles in shared memory until nothing
// changes anywhere (a flag in device memory, read by the host after every launch).
#include <cmath>
#include <vector>

#include "scene.h"

namespace {

constexpr uint8_t kInterior = 1, kBoundary = 2, kObstacle = 4;

// OR over the layers [k0, k1] of occupancy >= threshold
__global__ void k_project(const uint8_t* __restrict__ occ, int nx, int ny, int k0, int k1, uint8_t thr,
                          uint8_t* __restrict__ out) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y;
  if (x >= nx || y >= ny) return;
  uint8_t v = 0;
  for (int k = k0; k <= k1; ++k) v |= occ[((size_t)k * ny + y) * nx + x] >= thr ? 1 : 0;
  out[(size_t)y * nx + x] = v;
}

// 3x3 dilation (outside = 0) or erosion (outside = 1)
template <bool ERODE>
__global__ void k_morph(const uint8_t* __restrict__ in, int nx, int ny, uint8_t* __restrict__ out) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y;
  if (x >= nx || y >= ny) return;
  uint8_t v = ERODE ? 1 : 0;
  for (int dy = -1; dy <= 1; ++dy)
    for (int dx = -1; dx <= 1; ++dx) {
      const int xx = x + dx, yy = y + dy;
      const uint8_t p = (xx < 0 || xx >= nx || yy < 0 || yy >= ny) ? (ERODE ? 1 : 0) : in[(size_t)yy * nx + xx];
      v = ERODE ? (v & p) : (v | p);
    }
  out[(size_t)y * nx + x] = v;
}

// one flood-fill launch: every 32x32 tile (with a one-cell halo) is relaxed to its local fixed point
__global__ void __launch_bounds__(1024) k_fill(const uint8_t* __restrict__ wall, int nx, int ny,
                                               uint8_t* __restrict__ inside, int* __restrict__ changed) {
  __shared__ uint8_t s[34][34];
  __shared__ int again;
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int x = blockIdx.x * 32 + tx, y = blockIdx.y * 32 + ty;
  auto load = [&](int gx, int gy) -> uint8_t {
    return (gx < 0 || gx >= nx || gy < 0 || gy >= ny) ? 0 : inside[(size_t)gy * nx + gx];
  };
  s[ty + 1][tx + 1] = load(x, y);
  if (ty == 0) { s[0][tx + 1] = load(x, y - 1); s[33][tx + 1] = load(x, blockIdx.y * 32 + 32); }
  if (tx == 0) { s[ty + 1][0] = load(x - 1, y); s[ty + 1][33] = load(blockIdx.x * 32 + 32, y); }
  const bool is_free = x < nx && y < ny && !wall[(size_t)y * nx + x];
  bool mine = s[ty + 1][tx + 1] != 0, grew = false;
  __syncthreads();
  do {
    __syncthreads();
    if (tx == 0 && ty == 0) again = 0;
    __syncthreads();
    if (is_free && !mine && (s[ty][tx + 1] | s[ty + 2][tx + 1] | s[ty + 1][tx] | s[ty + 1][tx + 2])) {
      mine = true;
      grew = true;
      s[ty + 1][tx + 1] = 1;
      again = 1;
    }
    __syncthreads();
  } while (again);
  if (grew) {
    inside[(size_t)y * nx + x] = 1;
    *changed = 1;
  }
}

__global__ void k_plan(const uint8_t* __restrict__ inside, const uint8_t* __restrict__ low, int nx, int ny,
                       uint8_t* __restrict__ plan) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y * blockDim.y + threadIdx.y;
  if (x >= nx || y >= ny) return;
  auto in = [&](int gx, int gy) -> bool {
    return !(gx < 0 || gx >= nx || gy < 0 || gy >= ny) && inside[(size_t)gy * nx + gx];
  };
  uint8_t v = 0;
  if (in(x, y)) {
    v = kInterior;
    if (!(in(x - 1, y) && in(x + 1, y) && in(x, y - 1) && in(x, y + 1))) v |= kBoundary;
    if (low[(size_t)y * nx + x]) v |= kObstacle;
  }
  plan[(size_t)y * nx + x] = v;
}

// F1: layers whose centre fraction (k + 0.5)/nz lies in [lo, hi], binary64; returns false if none
bool slice_range(int nz, double lo, double hi, int& k0, int& k1) {
  k0 = nz; k1 = -1;
  for (int k = 0; k < nz; ++k) {
    const double c = ((double)k + 0.5) / (double)nz;
    if (lo <= c && c <= hi) { if (k < k0) k0 = k; k1 = k; }
  }
  return k1 >= k0;
}

}  // namespace

extern "C" r360_status r360_floorplan(const int32_t dims[3], const uint8_t* occupancy, uint8_t occ_threshold,
                                      int32_t seed_x, int32_t seed_y, const float upper[2], const float lower[2],
                                      uint8_t* plan_out) {
  if (!dims || !occupancy || !plan_out || occ_threshold < 1) return R360_ERR_INVALID_ARG;
  for (int a = 0; a < 3; ++a)
    if (dims[a] < 1) return R360_ERR_INVALID_ARG;
  const int nx = dims[0], ny = dims[1], nz = dims[2];
  if (seed_x < 0 || seed_x >= nx || seed_y < 0 || seed_y >= ny) return R360_ERR_INVALID_ARG;
  const double up_lo = upper ? (double)upper[0] : 0.60, up_hi = upper ? (double)upper[1] : 0.65;
  const double lo_lo = lower ? (double)lower[0] : 0.20, lo_hi = lower ? (double)lower[1] : 0.30;
  if (!(up_lo <= up_hi) || !(lo_lo <= lo_hi) || !std::isfinite(up_lo + up_hi + lo_lo + lo_hi)) return R360_ERR_INVALID_ARG;
  const size_t n2 = (size_t)nx * ny, N = n2 * nz;
  uint8_t *d_occ = nullptr, *d_a = nullptr, *d_b = nullptr, *d_low = nullptr, *d_in = nullptr;
  int* d_changed = nullptr;
  r360_status rc = R360_OK;
#define F_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { rc = r360_cuda_fail(e_, #call); goto done; } } while (0)
  {
    const dim3 blk(32, 8), grd((nx + 31) / 32, (ny + 7) / 8);
    const dim3 fblk(32, 32), fgrd((nx + 31) / 32, (ny + 31) / 32);
    int k0, k1;
    uint8_t seed_wall = 0, one = 1;
    F_CUDA(cudaMalloc(&d_occ, N));
    F_CUDA(cudaMalloc(&d_a, n2));
    F_CUDA(cudaMalloc(&d_b, n2));
    F_CUDA(cudaMalloc(&d_low, n2));
    F_CUDA(cudaMalloc(&d_in, n2));
    F_CUDA(cudaMalloc(&d_changed, sizeof(int)));
    F_CUDA(cudaMemcpy(d_occ, occupancy, N, cudaMemcpyHostToDevice));
    // F2 upper projection -> d_a ; F3 closing: dilate -> d_b, erode -> d_a (= wall)
    if (slice_range(nz, up_lo, up_hi, k0, k1)) k_project<<<grd, blk>>>(d_occ, nx, ny, k0, k1, occ_threshold, d_a);
    else F_CUDA(cudaMemset(d_a, 0, n2));
    k_morph<false><<<grd, blk>>>(d_a, nx, ny, d_b);
    k_morph<true><<<grd, blk>>>(d_b, nx, ny, d_a);
    if (slice_range(nz, lo_lo, lo_hi, k0, k1)) k_project<<<grd, blk>>>(d_occ, nx, ny, k0, k1, occ_threshold, d_low);
    else F_CUDA(cudaMemset(d_low, 0, n2));
    F_CUDA(cudaGetLastError());
    F_CUDA(cudaMemcpy(&seed_wall, d_a + (size_t)seed_y * nx + seed_x, 1, cudaMemcpyDeviceToHost));
    if (seed_wall) { rc = R360_ERR_INVALID_ARG; goto done; }      // the seed must be a free cell
    // F4 flood fill from the seed
    F_CUDA(cudaMemset(d_in, 0, n2));
    F_CUDA(cudaMemcpy(d_in + (size_t)seed_y * nx + seed_x, &one, 1, cudaMemcpyHostToDevice));
    // every launch relaxes each 32 x 32 tile to its local fixed point; a launch that changes anything adds at
    // least one cell, so the fill ends after at most nx * ny launches -- it runs until nothing changes (a winding
    // free region crosses tile borders far more often than any bound in nx + ny allows: ADVICE round 1)
    {
      int changed = 1;
      for (size_t it = 0; changed; ++it) {
        if (it > n2 + 8) { rc = R360_ERR_CUDA; goto done; }
        F_CUDA(cudaMemset(d_changed, 0, sizeof(int)));
        k_fill<<<fgrd, fblk>>>(d_a, nx, ny, d_in, d_changed);
        F_CUDA(cudaMemcpy(&changed, d_changed, sizeof(int), cudaMemcpyDeviceToHost));
      }
    }
    // F5-F7
    k_plan<<<grd, blk>>>(d_in, d_low, nx, ny, d_b);
    F_CUDA(cudaGetLastError());
    F_CUDA(cudaMemcpy(plan_out, d_b, n2, cudaMemcpyDeviceToHost));
  }
done:
#undef F_CUDA
  cudaFree(d_occ); cudaFree(d_a); cudaFree(d_b); cudaFree(d_low); cudaFree(d_in); cudaFree(d_changed);
  return rc;
}
