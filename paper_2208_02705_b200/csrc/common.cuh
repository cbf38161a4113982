// r360 -- shared device-side declarations of the CUDA path (sm_100a).
// Nothing here is shared with oracle/ (which is plain C and has its own header).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace r360 {

// Fused occupancy + label grid (uint16 per voxel):
//   value <  kEmptyBase : occupied, the value is the subfield label
//   value >= kEmptyBase : empty
// and, beside it, the skip distances of the empty voxels, ONE PER OCTANT of ray directions (uint8[N][8], octant
// o = [d_x < 0] + 2 [d_y < 0] + 4 [d_z < 0]): skip[v][o] = min(255, largest D such that the cube of D voxels per axis
// that starts at v and extends in the octant's direction holds no occupied voxel) >= 1 for an empty v.  A ray only
// ever moves forward on every axis, so this one-sided cube is all it can reach before it leaves it -- and it is far
// larger than a cube centred on v (next to a wall a ray that leaves the wall jumps the whole room, where the
// distance to the NEAREST occupied voxel is 1).
constexpr uint32_t kEmptyBase = 0xFF00u;
constexpr int kMaxSubfields = 0xFF00;
constexpr int kTileRows = 128;              // rows (samples) per MLP tile
constexpr float kParallelEps = 7.888609052210118e-31f;  // 2^-100: |d_a| below = axis-parallel (reading C1)

// Geometry of the grid, passed by value to kernels.
struct GridParams {
  int dims[3];
  float box_min[3];
  float vs[3];           // voxel size per axis: (box_max - box_min) / dims, binary32 (reading C)
  float inv_vs[3];       // 1 / vs: only for index GUESSES that are then verified against the planes
  const uint8_t* skip;   // device, [N][8]: octant skip distances of the empty voxels (above); REQUIRED by the Walker (never
                         // null: r360_scene_create always builds it; the fusion walk in fuse.cu does not use the Walker)
  int K;                 // samples per occupied voxel crossed (reading D)
  float Kf;
  float Kinv;            // 1 / K when K is a power of two (x * Kinv is then x / K bit for bit), else 0
};

// delta = (t_out - t_in) / K (reading D).  For a power of two the product with the exact reciprocal is the same
// correctly rounded value as the quotient and costs one instruction instead of the division sequence.
__device__ __forceinline__ float seg_delta(const GridParams& g, float t_in, float t_out) {
  const float w = __fsub_rn(t_out, t_in);
  return g.Kinv != 0.0f ? __fmul_rn(w, g.Kinv) : __fdiv_rn(w, g.Kf);
}

// One frame (or chunk) of rays.  ray id r (chunk-relative) -> global ray = ray0 + r;
// pose b = global / (W*H), pixel = global % (W*H), j = pixel / W, i = pixel % W.
struct FrameParams {
  int W, H;
  long long ray0;        // first global ray of this chunk
  long long out0;        // index of the chunk's first ray in the caller's output buffers (ray0 - first ray of the call)
  int out_format;        // r360_output_format: 0 = rgb float[3] + depth float, 1 = rgb uint8[3] + depth binary16
  unsigned pose0;        // ray0 / (W*H)
  unsigned pix0;         // ray0 % (W*H)
  unsigned n_rays;       // rays in this chunk
  int camera;            // 0 equirect (Eq.2-3), 1 pinhole (reading P)
  const float* poses;    // device [B*12]
  const float* sin_phi;  // device [W]  (reading B2: host binary64 libm, rounded once); pinhole: x_i
  const float* cos_phi;
  const float* sin_theta;  // device [H]; pinhole: y_j
  const float* cos_theta;
};

// Binned segment record: one occupied voxel crossed by one ray (K samples), 32 bytes = two uint4:
//   [0]: x = chunk-relative ray id, y = bits of t_in, z = bits of delta, w = ray-major segment slot
//   [1]: bits of the ray direction d.x, d.y, d.z, and the pose index (so that the MLP kernels need no per-ray
//        work and one address computation fetches everything a sample row needs)
typedef uint4 SegRec;
constexpr int kRecWords = 2;              // uint4 per record

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
  float x, y, z;
  if (f.camera == 0) {
    float sp = __ldg(f.sin_phi + i), cp = __ldg(f.cos_phi + i);
    float st = __ldg(f.sin_theta + j), ct = __ldg(f.cos_theta + j);
    x = __fmul_rn(ct, sp);
    y = -st;
    z = __fmul_rn(ct, cp);
  } else {
    // reading P: d_cam = (x, y, 1)/|(x, y, 1)|, n2 = (x*x + y*y) + 1, inv = 1/sqrt(n2), each operation rounded
    const float px = __ldg(f.sin_phi + i), py = __ldg(f.sin_theta + j);
    const float n2 = __fadd_rn(__fadd_rn(__fmul_rn(px, px), __fmul_rn(py, py)), 1.0f);
    const float inv = __fdiv_rn(1.0f, __fsqrt_rn(n2));
    x = __fmul_rn(px, inv);
    y = __fmul_rn(py, inv);
    z = inv;
  }
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
// Voxel walk (readings C1-C4) with exact empty-space skipping.  next() advances to the next OCCUPIED
// voxel the ray crosses (t_in < t_out, strict), front to back, and returns false when the ray has
// left the grid.
//
// Reading C5: the crossed set is a per-voxel predicate, max(t0, max_a tn_a(i)) < min_a tf_a(i), with
// every distance computed from the voxel index through t_at(); it does not depend on the path taken.
// So from an empty voxel whose skip distance (for the ray's octant) is D the walk leaves the whole empty
// cube [idx, idx + (D-1) step] at once: the exit distance `to` is the smallest far-plane distance of the
// CUBE, the axis of the minimum steps to the voxel behind that plane, and on the other two axes the new
// index is the first one (along the ray) whose far plane lies beyond `to` -- found from a position guess
// that is checked against the planes themselves (a too large guess is walked back here, a too small one
// corrects itself in the next iteration, see advance()), so no rounding of the guess can change the result.
// The entry distance of the next voxel is max(t0, to, its near planes), which is exactly the
// oracle's max(t0, tn_x, tn_y, tn_z); for a plain one-voxel step this reduces to max(ti, to).
struct Walker {
  float o[3], d[3], inv[3];
  float t0, ti;     // clip distance; entry distance of the current voxel
  int idx[3];
  int step[3], off[3];   // direction of travel per axis: step = +1 / -1, off = 1 / 0 (index offset of the far plane)
  int octant;            // [d_x < 0] + 2 [d_y < 0] + 4 [d_z < 0]: which skip distance of a voxel this ray uses
  bool par[3];
  bool alive;

  __device__ __forceinline__ float t_at(const GridParams& g, int a, int k) const {
    return __fmul_rn(__fsub_rn(plane(g, a, k), o[a]), inv[a]);
  }

  __device__ __forceinline__ void init(const GridParams& g, const Ray& ray) {
    alive = true;
    octant = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      o[a] = ray.o[a];
      d[a] = ray.d[a];
      par[a] = fabsf(ray.d[a]) < kParallelEps;
      off[a] = ray.d[a] < 0.0f ? 0 : 1;
      step[a] = 2 * off[a] - 1;
      octant |= (1 - off[a]) << a;
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
        float n_ = t_at(g, a, off[a] ? 0 : N);
        float f_ = t_at(g, a, off[a] ? N : 0);
        if (n_ > t0) t0 = n_;
        if (f_ < t1) t1 = f_;
      }
    }
    if (!(t0 < t1)) alive = false;
    // C3: start voxel; C4: its entry distance
    ti = t0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      float pa = __fmaf_rn(t0, ray.d[a], o[a]);
      float f = floorf(__fdiv_rn(__fsub_rn(pa, g.box_min[a]), g.vs[a]));
      int N = g.dims[a];
      idx[a] = (f < 0.0f) ? 0 : ((f > (float)(N - 1)) ? N - 1 : (int)f);
      if (!par[a]) ti = fmaxf(ti, t_at(g, a, idx[a] + 1 - off[a]));
    }
    // from here on a parallel axis never limits the walk: (plane - (-inf)) * 1 = +inf without a select
#pragma unroll
    for (int a = 0; a < 3; ++a)
      if (par[a]) { o[a] = __int_as_float(0xff800000); inv[a] = 1.0f; }
  }

  // One iteration of the walk (the ray must be alive): on true the voxel just left was an occupied crossed voxel,
  // lab = its subfield label, [t_in, t_out] its crossing interval.
  __device__ __forceinline__ bool advance(const GridParams& g, const uint16_t* __restrict__ grid,
                                       uint32_t& lab, float& t_in, float& t_out) {
    {
      // (unsigned index arithmetic: one multiply-add per level and a 32-bit offset)
      const uint32_t lin = ((uint32_t)idx[2] * (uint32_t)g.dims[1] + (uint32_t)idx[1]) * (uint32_t)g.dims[0] + (uint32_t)idx[0];
      const uint32_t l = __ldg(grid + lin);
      const uint32_t sk = __ldg(g.skip + (size_t)lin * 8u + (uint32_t)octant);   // requested with the grid word
      const bool empty = l >= kEmptyBase;
      const int r = empty ? (int)sk - 1 : 0;     // the cube [idx, idx + r step] is empty (0: this voxel only)
      // far planes of that cube, clamped to the grid
      int kx[3];
      float tf[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        kx[a] = min(max(idx[a] + step[a] * r + off[a], 0), g.dims[a]);
        tf[a] = t_at(g, a, kx[a]);
      }
      int amin = 2;
      float to = tf[2];
      if (tf[1] <= to) { to = tf[1]; amin = 1; }
      if (tf[0] <= to) { to = tf[0]; amin = 0; }   // ties -> lowest axis
      const bool hit = !empty && ti < to;
      if (hit) { lab = l; t_in = ti; t_out = to; }
      // step across the far plane of the axis of the minimum
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        if (a == amin) {
          idx[a] = kx[a] + off[a] - 1;
          if ((unsigned)idx[a] >= (unsigned)g.dims[a]) alive = false;
        }
      }
      if (r > 0) {
        // left a cube: re-derive the index on the other axes from the planes
        float tin = fmaxf(t0, to);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          if (a != amin && !par[a] && alive) {
            // the ray only moves forward: its index on this axis lies between idx and idx + r step
            const int lo = off[a] ? idx[a] : max(idx[a] - r, 0), hi = off[a] ? min(idx[a] + r, g.dims[a] - 1) : idx[a];
            const int first = idx[a];
            const float p = __fmaf_rn(to, d[a], o[a]);
            int gi = __float2int_rd((p - g.box_min[a]) * g.inv_vs[a]);     // guess; a too large one is corrected below
            gi = min(max(gi, lo), hi);
            // (A guess that is too SMALL needs no check here.  The voxel it names is then left at or before `to`:
            // its far plane on this axis is <= to <= the entry distance set below, so the next iteration finds
            // t_in >= t_out for it -- not crossed, nothing emitted, whatever it holds -- and steps across that
            // very plane with the entry distance unchanged; if it is empty with a skip cube, the cube holds the
            // ray's true voxel and is empty, so leaving it at once is as valid.  One plane distance per axis less
            // in every cube exit, one cheap extra iteration when the guess was off.)
            // backward: no earlier index of the cube may qualify; tn = near plane of gi
            float tn = t_at(g, a, gi - step[a] + off[a]);
            while (gi != first && tn > to) {
              gi -= step[a];
              tn = t_at(g, a, gi - step[a] + off[a]);
            }
            idx[a] = gi;
            tin = fmaxf(tin, tn);
          }
        }
        ti = tin;
      } else {
        ti = fmaxf(ti, to);
      }
      return hit;
    }
  }

  // Advances to the next OCCUPIED crossed voxel; false when the ray has left the grid.
  __device__ __forceinline__ bool next(const GridParams& g, const uint16_t* __restrict__ grid,
                                       uint32_t& lab, float& t_in, float& t_out) {
    while (alive)
      if (advance(g, grid, lab, t_in, t_out)) return true;
    return false;
  }
};

}  // namespace r360
