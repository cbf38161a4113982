// r360 -- shared device-side declarations of the CUDA path (sm_100a).
// Nothing here is shared with oracle/ (which is plain C and has its own header).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace r360 {

constexpr uint32_t kEmptyVoxel = 0xFFFFu;   // fused occupancy+label grid: 0xFFFF = empty
constexpr int kTileRows = 128;              // rows (samples) per MLP tile
constexpr float kParallelEps = 7.888609052210118e-31f;  // 2^-100: |d_a| below = axis-parallel (reading C1)

// Geometry of the grid, passed by value to kernels.
struct GridParams {
  int dims[3];
  float box_min[3];
  float vs[3];           // voxel size per axis: (box_max - box_min) / dims, binary32 (reading C)
  int K;                 // samples per occupied voxel crossed (reading D)
  float Kf;
};

// One frame (or chunk) of rays.  ray id r (chunk-relative) -> global ray = ray0 + r;
// pose b = global / (W*H), pixel = global % (W*H), j = pixel / W, i = pixel % W.
struct FrameParams {
  int W, H;
  long long ray0;        // first global ray of this chunk
  unsigned pose0;        // ray0 / (W*H)
  unsigned pix0;         // ray0 % (W*H)
  unsigned n_rays;       // rays in this chunk
  const float* poses;    // device [B*12]
  const float* sin_phi;  // device [W]  (reading B2: host binary64 libm, rounded once)
  const float* cos_phi;
  const float* sin_theta;  // device [H]
  const float* cos_theta;
};

// Binned segment record: one occupied voxel crossed by one ray (K samples).
//   x = chunk-relative ray id, y = bits of t_in, z = bits of delta, w = ray-major segment slot
typedef uint4 SegRec;

// ---------------------------------------------------------------------------------------
// Ray of a pixel.  Eq.3 and reading B3: every operation individually
// rounded (the __f*_rn intrinsics are never contracted into FMAs).
struct Ray {
  float o[3], d[3];
  unsigned pose;         // index into FrameParams::poses
};

__device__ __forceinline__ Ray make_ray(const FrameParams& f, unsigned r) {
  // 32-bit index math: a chunk never spans more than 2^31 rays and W*H < 2^31
  const unsigned wh = (unsigned)f.W * (unsigned)f.H;
  unsigned pix = f.pix0 + r;
  unsigned b = pix / wh;
  pix -= b * wh;
  b += f.pose0;
  const unsigned j = pix / (unsigned)f.W;
  const unsigned i = pix - j * (unsigned)f.W;
  const float* P = f.poses + b * 12;
  float sp = __ldg(f.sin_phi + i), cp = __ldg(f.cos_phi + i);
  float st = __ldg(f.sin_theta + j), ct = __ldg(f.cos_theta + j);
  float x = __fmul_rn(ct, sp);
  float y = -st;
  float z = __fmul_rn(ct, cp);
  Ray ray;
  ray.pose = b;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float m0 = __fmul_rn(__ldg(P + a * 4 + 0), x);
    float m1 = __fmul_rn(__ldg(P + a * 4 + 1), y);
    float m2 = __fmul_rn(__ldg(P + a * 4 + 2), z);
    ray.d[a] = __fadd_rn(__fadd_rn(m0, m1), m2);
    ray.o[a] = __ldg(P + a * 4 + 3);
  }
  return ray;
}

// Plane k of axis a: box_min + k*s, one multiply, one add (reading C).
__device__ __forceinline__ float plane(const GridParams& g, int a, int k) {
  return __fadd_rn(g.box_min[a], __fmul_rn((float)k, g.vs[a]));
}

// ---------------------------------------------------------------------------------------
// Voxel walk (readings C1-C4) as a resumable state machine.  next() advances to the next
// OCCUPIED voxel the ray crosses (t_in < t_out, strict), front to back, and returns false when
// the ray has left the grid.  Distances always come from the voxel index through t_at(); only
// the axis that stepped is recomputed, and the new near distance of that axis is the old far
// distance (same formula, same index => same bits as recomputing it).
struct Walker {
  float o[3], inv[3];
  float tn[3], tf[3];
  float t0;
  int idx[3];
  int v;            // linear voxel index
  bool neg[3];
  bool alive;

  __device__ __forceinline__ float t_at(const GridParams& g, int a, int k) const {
    return __fmul_rn(__fsub_rn(plane(g, a, k), o[a]), inv[a]);
  }

  __device__ __forceinline__ void init(const GridParams& g, const Ray& ray) {
    bool par[3];
    alive = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      o[a] = ray.o[a];
      par[a] = fabsf(ray.d[a]) < kParallelEps;
      neg[a] = ray.d[a] < 0.0f;
      inv[a] = par[a] ? 0.0f : __fdiv_rn(1.0f, ray.d[a]);
    }
    // C2: clip against the box
    t0 = 0.0f;
    float t1 = __int_as_float(0x7f800000);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      int N = g.dims[a];
      if (par[a]) {
        if (!(o[a] >= g.box_min[a] && o[a] < plane(g, a, N))) alive = false;
      } else {
        float n_ = t_at(g, a, neg[a] ? N : 0);
        float f_ = t_at(g, a, neg[a] ? 0 : N);
        if (n_ > t0) t0 = n_;
        if (f_ < t1) t1 = f_;
      }
    }
    if (!(t0 < t1)) alive = false;
    // C3: start voxel
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      float pa = __fmaf_rn(t0, ray.d[a], o[a]);
      float f = floorf(__fdiv_rn(__fsub_rn(pa, g.box_min[a]), g.vs[a]));
      int N = g.dims[a];
      idx[a] = (f < 0.0f) ? 0 : ((f > (float)(N - 1)) ? N - 1 : (int)f);
      if (par[a]) {
        tn[a] = __int_as_float(0xff800000);
        tf[a] = __int_as_float(0x7f800000);
      } else {
        tn[a] = t_at(g, a, idx[a] + (neg[a] ? 1 : 0));
        tf[a] = t_at(g, a, idx[a] + (neg[a] ? 0 : 1));
      }
    }
    v = (idx[2] * g.dims[1] + idx[1]) * g.dims[0] + idx[0];
  }

  // C4.  On true: lab = subfield label of the voxel, [t_in, t_out] its crossing interval.
  __device__ __forceinline__ bool next(const GridParams& g, const uint16_t* __restrict__ grid,
                                       uint32_t& lab, float& t_in, float& t_out) {
    while (alive) {
      float ti = fmaxf(fmaxf(t0, tn[0]), fmaxf(tn[1], tn[2]));
      int amin = 2;
      float to = tf[2];
      if (tf[1] <= to) { to = tf[1]; amin = 1; }
      if (tf[0] <= to) { to = tf[0]; amin = 0; }   // ties -> lowest axis
      bool hit = false;
      if (ti < to) {
        uint32_t l = __ldg(grid + v);
        if (l != kEmptyVoxel) { hit = true; lab = l; t_in = ti; t_out = to; }
      }
      // advance along amin (selects instead of dynamic register indexing)
      int stride = 1;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        if (a == amin) {
          int s = neg[a] ? -1 : 1;
          idx[a] += s;
          v += s * stride;
          tn[a] = tf[a];
          tf[a] = t_at(g, a, idx[a] + (neg[a] ? 0 : 1));
          if (idx[a] < 0 || idx[a] >= g.dims[a]) alive = false;
        }
        stride *= g.dims[a];
      }
      if (hit) return true;
    }
    return false;
  }
};

}  // namespace r360
