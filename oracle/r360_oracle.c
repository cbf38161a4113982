/* r360 ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See r360_oracle.h.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fopenmp -fPIC -shared
 * Every function cites the passage of /root/reference/PAPER.md (or the DESIGN.md
 * reading) it follows.  No blocking, fusion or reordering beyond those.
 */
#include "r360_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define R360O_PI 3.14159265358979323846

struct r360o_scene {
  r360o_desc d;
  int64_t n_vox;
  int64_t P;            /* parameters per subfield */
  float vs[3];          /* voxel size per axis, binary32: (box_max-box_min)/dims (C) */
  uint8_t* occ;
  int32_t* label;
  float* w;             /* n*P */
  float* centre;        /* n*3 (A3) */
  float* inv_half;      /* n*3 (A3) */
  int32_t cam_model;    /* 0 = equirectangular (Eq.2-3), 1 = pinhole (reading P) */
  double fx, fy, cx, cy;
};

/* ---------------------------------------------------------------- layout (A1)
 * PAPER.md:413 "6212 parameters", :200 "4 fully-connected 32-channel layers",
 * Table 4 :434-444.  Blob per subfield, W[out][in] row-major then b[out]:
 * trunk-1 (Wd x pe_p), trunk-2..Hd (Wd x Wd), density (1 x Wd), feature (Wd x Wd),
 * colour (Wd x (Wd+pe_d)), rgb (3 x Wd). */
static int pe_dim(int L) { return 3 + 6 * L; }

int64_t r360o_params_per_subfield(const r360o_desc* d) {
  int64_t Wd = d->hidden_width, pp = pe_dim(d->pe_pos_levels), pd = pe_dim(d->pe_dir_levels);
  int64_t P = Wd * pp + Wd;
  P += (int64_t)(d->n_hidden - 1) * (Wd * Wd + Wd);
  P += Wd + 1;
  P += Wd * Wd + Wd;
  P += Wd * (Wd + pd) + Wd;
  P += 3 * Wd + 3;
  return P;
}

/* Plane k of axis a (C): box_min + k*s, one multiply and one add, each rounded. */
static float plane(const r360o_scene* s, int a, int k) {
  float ks = (float)k * s->vs[a];
  return s->d.box_min[a] + ks;
}

r360o_scene* r360o_create(const r360o_desc* desc, const uint8_t* occupancy,
                          const int32_t* voxel_subfield, const float* weights) {
  if (!desc || !occupancy || !voxel_subfield || !weights) return NULL;
  for (int a = 0; a < 3; ++a) {
    if (desc->dims[a] < 1) return NULL;
    if (!(desc->box_max[a] > desc->box_min[a])) return NULL;
  }
  if (desc->n_subfields < 1 || desc->hidden_width < 1 || desc->n_hidden < 1) return NULL;
  if (desc->pe_pos_levels < 0 || desc->pe_dir_levels < 0 || desc->samples_per_voxel < 1) return NULL;
  r360o_scene* s = (r360o_scene*)calloc(1, sizeof(*s));
  s->d = *desc;
  s->n_vox = (int64_t)desc->dims[0] * desc->dims[1] * desc->dims[2];
  s->P = r360o_params_per_subfield(desc);
  for (int a = 0; a < 3; ++a) {
    float ext = desc->box_max[a] - desc->box_min[a];
    s->vs[a] = ext / (float)desc->dims[a];
  }
  int64_t n = desc->n_subfields;
  s->occ = (uint8_t*)malloc((size_t)s->n_vox);
  s->label = (int32_t*)malloc((size_t)s->n_vox * sizeof(int32_t));
  s->w = (float*)malloc((size_t)(n * s->P) * sizeof(float));
  s->centre = (float*)calloc((size_t)n * 3, sizeof(float));
  s->inv_half = (float*)calloc((size_t)n * 3, sizeof(float));
  memcpy(s->occ, occupancy, (size_t)s->n_vox);
  memcpy(s->label, voxel_subfield, (size_t)s->n_vox * sizeof(int32_t));
  memcpy(s->w, weights, (size_t)(n * s->P) * sizeof(float));
  /* A3: axis-aligned bounding box (voxel faces) of each subfield's voxels */
  int32_t* lo = (int32_t*)malloc((size_t)n * 3 * sizeof(int32_t));
  int32_t* hi = (int32_t*)malloc((size_t)n * 3 * sizeof(int32_t));
  for (int64_t k = 0; k < n * 3; ++k) { lo[k] = INT32_MAX; hi[k] = -1; }
  int bad = 0;
  for (int64_t v = 0; v < s->n_vox; ++v) {
    if (s->occ[v] < desc->occ_threshold) continue;
    int32_t k = s->label[v];
    if (k < 0 || k >= n) { bad = 1; break; }
    int32_t idx[3];
    idx[0] = (int32_t)(v % desc->dims[0]);
    idx[1] = (int32_t)((v / desc->dims[0]) % desc->dims[1]);
    idx[2] = (int32_t)(v / ((int64_t)desc->dims[0] * desc->dims[1]));
    for (int a = 0; a < 3; ++a) {
      if (idx[a] < lo[k * 3 + a]) lo[k * 3 + a] = idx[a];
      if (idx[a] > hi[k * 3 + a]) hi[k * 3 + a] = idx[a];
    }
  }
  for (int64_t k = 0; k < n && !bad; ++k) {
    for (int a = 0; a < 3; ++a) {
      if (hi[k * 3 + a] < 0) { /* subfield owns no voxel: never sampled */
        s->centre[k * 3 + a] = 0.0f;
        s->inv_half[k * 3 + a] = 1.0f;
        continue;
      }
      float pl = plane(s, a, lo[k * 3 + a]);
      float ph = plane(s, a, hi[k * 3 + a] + 1);
      float sum = pl + ph;
      float dif = ph - pl;
      float c = 0.5f * sum;
      float h = 0.5f * dif;
      s->centre[k * 3 + a] = c;
      s->inv_half[k * 3 + a] = 1.0f / h;
    }
  }
  free(lo);
  free(hi);
  for (int64_t i = 0; i < n * s->P && !bad; ++i)
    if (!isfinite(s->w[i])) bad = 1;
  if (bad) { r360o_destroy(s); return NULL; }
  return s;
}

void r360o_destroy(r360o_scene* s) {
  if (!s) return;
  free(s->occ); free(s->label); free(s->w); free(s->centre); free(s->inv_half);
  free(s);
}

/* ---------------------------------------------------------------- rays (B) */

/* Reading B1: pixel centres.  phi_i = (i + 0.5 - W/2) * 2pi/W ;
 * theta_j = -(j + 0.5 - H/2) * pi/H   (inverse of Eq.2). */
void r360o_pixel_to_sphere(int32_t i, int32_t j, int32_t W, int32_t H, double* phi, double* theta) {
  *phi = (((double)i + 0.5) - (double)W / 2.0) * (2.0 * R360O_PI / (double)W);
  *theta = -((((double)j + 0.5) - (double)H / 2.0) * (R360O_PI / (double)H));
}

/* Eq.2: u = phi*W/(2pi) + W/2 ; v = -theta*H/pi + H/2 */
void r360o_sphere_to_pixel(double phi, double theta, int32_t W, int32_t H, double* u, double* v) {
  *u = phi * (double)W / (2.0 * R360O_PI) + (double)W / 2.0;
  *v = -theta * (double)H / R360O_PI + (double)H / 2.0;
}

/* Reading B2: trig of the pixel-centre angles in binary64 libm, rounded once. */
void r360o_trig_tables(int32_t W, int32_t H, float* sin_phi, float* cos_phi,
                       float* sin_theta, float* cos_theta) {
  double phi, theta;
  for (int32_t i = 0; i < W; ++i) {
    r360o_pixel_to_sphere(i, 0, W, H, &phi, &theta);
    sin_phi[i] = (float)sin(phi);
    cos_phi[i] = (float)cos(phi);
  }
  for (int32_t j = 0; j < H; ++j) {
    r360o_pixel_to_sphere(0, j, W, H, &phi, &theta);
    sin_theta[j] = (float)sin(theta);
    cos_theta[j] = (float)cos(theta);
  }
}

/* Eq.3: (x,y,z) = (cos th sin ph, -sin th, cos th cos ph);
 * reading B3: d_a = (R_a0*x + R_a1*y) + R_a2*z, every operation rounded. */
static void ray_dir(const float pose[12], float sp, float cp, float st, float ct, float d[3]) {
  float x = ct * sp;
  float y = -st;
  float z = ct * cp;
  for (int a = 0; a < 3; ++a) {
    float m0 = pose[a * 4 + 0] * x;
    float m1 = pose[a * 4 + 1] * y;
    float m2 = pose[a * 4 + 2] * z;
    float s01 = m0 + m1;
    d[a] = s01 + m2;
  }
}

void r360o_ray(const float pose[12], int32_t W, int32_t H, int32_t i, int32_t j, float o[3], float d[3]) {
  double phi, theta;
  r360o_pixel_to_sphere(i, j, W, H, &phi, &theta);
  ray_dir(pose, (float)sin(phi), (float)cos(phi), (float)sin(theta), (float)cos(theta), d);
  o[0] = pose[3]; o[1] = pose[7]; o[2] = pose[11];
}

/* ---------------------------------------------------------------- pinhole view (reading P)
 * The paper shows "perspective views" while roaming (720p timings :200) and gives no
 * camera model.  Reading P: the standard pinhole in the camera frame of Eq.3 (x right, y down, z
 * forward): pixel centre (i+0.5, j+0.5) -> x = (i + 0.5 - cx)/fx, y = (j + 0.5 - cy)/fy,
 * binary64, rounded once to binary32 (tables, like B2); d_cam = (x, y, 1)/|(x, y, 1)| in binary32,
 * every operation rounded: n2 = (x*x + y*y) + 1, inv = 1/sqrt(n2), d_cam = (x*inv, y*inv, inv);
 * then d = R d_cam as in B3.  t stays the metric distance along the unit ray (as for the panorama). */
void r360o_pinhole_tables(int32_t W, int32_t H, double fx, double fy, double cx, double cy, float* x, float* y) {
  for (int32_t i = 0; i < W; ++i) x[i] = (float)((((double)i + 0.5) - cx) / fx);
  for (int32_t j = 0; j < H; ++j) y[j] = (float)((((double)j + 0.5) - cy) / fy);
}

static void pinhole_dir(const float pose[12], float x, float y, float d[3]) {
  float xx = x * x;
  float yy = y * y;
  float s2 = xx + yy;
  float n2 = s2 + 1.0f;
  float inv = 1.0f / sqrtf(n2);
  float c[3];
  c[0] = x * inv;
  c[1] = y * inv;
  c[2] = inv;
  for (int a = 0; a < 3; ++a) {
    float m0 = pose[a * 4 + 0] * c[0];
    float m1 = pose[a * 4 + 1] * c[1];
    float m2 = pose[a * 4 + 2] * c[2];
    float s01 = m0 + m1;
    d[a] = s01 + m2;
  }
}

void r360o_ray_pinhole(const float pose[12], double fx, double fy, double cx, double cy, int32_t i, int32_t j,
                       float o[3], float d[3]) {
  float x = (float)((((double)i + 0.5) - cx) / fx);
  float y = (float)((((double)j + 0.5) - cy) / fy);
  pinhole_dir(pose, x, y, d);
  o[0] = pose[3]; o[1] = pose[7]; o[2] = pose[11];
}

int r360o_set_camera(r360o_scene* s, int32_t model, double fx, double fy, double cx, double cy) {
  if (!s || (model != 0 && model != 1)) return 1;
  if (model == 1 && !(fx > 0.0 && fy > 0.0 && isfinite(fx) && isfinite(fy) && isfinite(cx) && isfinite(cy))) return 1;
  s->cam_model = model; s->fx = fx; s->fy = fy; s->cx = cx; s->cy = cy;
  return 0;
}

/* per-image tables of the scene's camera: 2W + 2H floats (equirect: sin/cos phi, sin/cos theta;
 * pinhole: x in the first W, y in the third block, the rest unused) and the direction of pixel (i,j) */
static float* camera_tables(const r360o_scene* s, int32_t W, int32_t H) {
  float* tab = (float*)calloc((size_t)(2 * W + 2 * H), sizeof(float));
  if (s->cam_model == 1) r360o_pinhole_tables(W, H, s->fx, s->fy, s->cx, s->cy, tab, tab + 2 * W);
  else r360o_trig_tables(W, H, tab, tab + W, tab + 2 * W, tab + 2 * W + H);
  return tab;
}

static void camera_dir(const r360o_scene* s, const float pose[12], const float* tab, int32_t W, int32_t H,
                       int i, int j, float d[3]) {
  if (s->cam_model == 1) pinhole_dir(pose, tab[i], tab[2 * W + j], d);
  else ray_dir(pose, tab[i], tab[W + i], tab[2 * W + j], tab[2 * W + H + j], d);
}

/* ---------------------------------------------------------------- traversal (C)
 * PAPER.md:174 "ray casting techniques to quickly localize occupied voxels";
 * :29 / :105 empty-space skipping. */

#define PARALLEL_EPS 7.888609052210118e-31f /* 2^-100: |d_a| below this = axis-parallel (C1) */

typedef struct {
  float o[3], d[3], inv[3];
  int par[3];   /* axis-parallel */
  int neg[3];   /* d_a < 0 */
} ray_t;

static void ray_setup(ray_t* r, const float o[3], const float d[3]) {
  for (int a = 0; a < 3; ++a) {
    r->o[a] = o[a];
    r->d[a] = d[a];
    r->par[a] = fabsf(d[a]) < PARALLEL_EPS;
    r->neg[a] = d[a] < 0.0f;
    r->inv[a] = r->par[a] ? 0.0f : 1.0f / d[a];
  }
}

/* C1: entry/exit distance of the slab [plane(k_near), plane(k_far)] on axis a */
static float t_at(const r360o_scene* s, const ray_t* r, int a, int k) {
  float diff = plane(s, a, k) - r->o[a];
  return diff * r->inv[a];
}

/* C2 */
static int clip(const r360o_scene* s, const ray_t* r, float* t0, float* t1) {
  float lo = 0.0f, hi = INFINITY;
  for (int a = 0; a < 3; ++a) {
    int N = s->d.dims[a];
    if (r->par[a]) {
      if (!(r->o[a] >= s->d.box_min[a] && r->o[a] < plane(s, a, N))) return 0;
      continue;
    }
    float tn = t_at(s, r, a, r->neg[a] ? N : 0);
    float tf = t_at(s, r, a, r->neg[a] ? 0 : N);
    if (tn > lo) lo = tn;
    if (tf < hi) hi = tf;
  }
  *t0 = lo;
  *t1 = hi;
  return lo < hi;
}

int r360o_clip(const r360o_scene* s, const float o[3], const float d[3], float* t0, float* t1) {
  ray_t r;
  ray_setup(&r, o, d);
  return clip(s, &r, t0, t1);
}

typedef void (*visit_fn)(void* ctx, int64_t voxel, float t_in, float t_out, int occupied);

/* C3-C4: walk, calling visit() for every crossed voxel (t_in < t_out, strict). */
static void walk(const r360o_scene* s, const ray_t* r, visit_fn visit, void* ctx) {
  float t0, t1;
  /* a direction with no component of 2^-100 or more (reading C1 makes every axis parallel) goes nowhere: it crosses
   * no voxel boundary and there is no exit axis to step along (reading B5 keeps such rays out of the render calls) */
  if (r->par[0] && r->par[1] && r->par[2]) return;
  if (!clip(s, r, &t0, &t1)) return;
  int idx[3];
  for (int a = 0; a < 3; ++a) {                       /* C3 */
    float pa = fmaf(t0, r->d[a], r->o[a]);
    float rel = pa - s->d.box_min[a];
    float f = floorf(rel / s->vs[a]);
    int N = s->d.dims[a];
    int i = (f < 0.0f) ? 0 : ((f > (float)(N - 1)) ? N - 1 : (int)f);
    idx[a] = i;
  }
  for (;;) {                                          /* C4 */
    float t_in = t0, t_out = INFINITY;
    int amin = -1;
    for (int a = 0; a < 3; ++a) {
      if (r->par[a]) continue;
      float tn = t_at(s, r, a, idx[a] + (r->neg[a] ? 1 : 0));
      float tf = t_at(s, r, a, idx[a] + (r->neg[a] ? 0 : 1));
      if (tn > t_in) t_in = tn;
      if (tf < t_out) { t_out = tf; amin = a; }       /* strict <: ties -> lowest axis */
    }
    if (t_in < t_out) {
      int64_t v = ((int64_t)idx[2] * s->d.dims[1] + idx[1]) * s->d.dims[0] + idx[0];
      visit(ctx, v, t_in, t_out, s->occ[v] >= s->d.occ_threshold);
    }
    idx[amin] += r->neg[amin] ? -1 : 1;
    if (idx[amin] < 0 || idx[amin] >= s->d.dims[amin]) break;
  }
}

typedef struct {
  int only_occ;
  int64_t cap, n;
  int32_t* voxel;
  float *t_in, *t_out;
} collect_t;

static void collect_visit(void* vctx, int64_t v, float t_in, float t_out, int occupied) {
  collect_t* c = (collect_t*)vctx;
  if (c->only_occ && !occupied) return;
  if (c->n < c->cap) {
    if (c->voxel) c->voxel[c->n] = (int32_t)v;
    if (c->t_in) c->t_in[c->n] = t_in;
    if (c->t_out) c->t_out[c->n] = t_out;
  }
  c->n++;
}

int64_t r360o_walk(const r360o_scene* s, const float o[3], const float d[3], int only_occupied,
                   int64_t cap, int32_t* voxel, float* t_in, float* t_out) {
  ray_t r;
  ray_setup(&r, o, d);
  collect_t c = {only_occupied, cap, 0, voxel, t_in, t_out};
  walk(s, &r, collect_visit, &c);
  return c.n;
}

/* ---------------------------------------------------------------- samples (D)
 * PAPER.md:164 "densely sample the occupied voxels instead of uniform sampling
 * along the rays"; reading D: K stratum midpoints per crossed occupied voxel. */
typedef struct {
  const r360o_scene* s;
  int64_t cap, n;
  float *t, *delta;
  int32_t* sid;
} sample_t;

static void sample_visit(void* vctx, int64_t v, float t_in, float t_out, int occupied) {
  sample_t* c = (sample_t*)vctx;
  if (!occupied) return;
  int K = c->s->d.samples_per_voxel;
  float len = t_out - t_in;
  float delta = len / (float)K;
  for (int j = 0; j < K; ++j) {
    if (c->n < c->cap) {
      c->t[c->n] = fmaf((float)j + 0.5f, delta, t_in);
      c->delta[c->n] = delta;
      c->sid[c->n] = c->s->label[v];
    }
    c->n++;
  }
}

static int64_t ray_samples(const r360o_scene* s, const float o[3], const float d[3], int64_t cap,
                           float* t, float* delta, int32_t* sid) {
  ray_t r;
  ray_setup(&r, o, d);
  sample_t c = {s, cap, 0, t, delta, sid};
  walk(s, &r, sample_visit, &c);
  return c.n;
}

/* Reading B5: a pose is admissible iff its 12 entries are finite and its 3x3 part M, taken in binary64,
 * has 2^-16 <= |M|_F <= 2^16 and |det M| >= 2^-16 |M|_F^3.  Every rotation passes (|det| / |M|_F^3 = 3^-1.5 = 0.19),
 * also with a moderate scale; a singular or nearly singular M, which maps some unit camera direction of Eq. 3 to
 * (nearly) zero, does not: the smallest singular value of an admissible M is at least |det| / |M|_F^2 >=
 * 2^-16 |M|_F, far above the rounding of reading B3's three products and two sums (about 2^-22 |M|_F). */
int r360o_pose_ok(const float pose[12]) {
  if (!pose) return 0;
  for (int a = 0; a < 12; ++a) if (!isfinite(pose[a])) return 0;
  double m[3][3], f2 = 0.0;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) { m[a][b] = (double)pose[a * 4 + b]; f2 += m[a][b] * m[a][b]; }
  double f = sqrt(f2);
  double det = m[0][0] * (m[1][1] * m[2][2] - m[1][2] * m[2][1]) - m[0][1] * (m[1][0] * m[2][2] - m[1][2] * m[2][0]) +
               m[0][2] * (m[1][0] * m[2][1] - m[1][1] * m[2][0]);
  const double lim = 1.0 / 65536.0;
  if (!(f >= lim && f <= 65536.0)) return 0;
  return fabs(det) >= lim * f * f * f;
}

int64_t r360o_ray_samples(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                          int32_t i, int32_t j, int64_t cap, float* t, float* delta, int32_t* subfield) {
  float o[3], d[3];
  if (!r360o_pose_ok(pose)) return -2;
  if (s->cam_model == 1) r360o_ray_pinhole(pose, s->fx, s->fy, s->cx, s->cy, i, j, o, d);
  else r360o_ray(pose, W, H, i, j, o, d);
  return ray_samples(s, o, d, cap, t, delta, subfield);
}

/* ---------------------------------------------------------------- field (A, F) */

void r360o_subfield_frame(const r360o_scene* s, int32_t k, float centre[3], float inv_half[3]) {
  for (int a = 0; a < 3; ++a) {
    centre[a] = s->centre[(int64_t)k * 3 + a];
    inv_half[a] = s->inv_half[(int64_t)k * 3 + a];
  }
}

/* A2 (Eq.1, "applied individually on each component"):
 * F(x) = [x, sin(2^0 x), cos(2^0 x), ..., sin(2^(L-1) x), cos(2^(L-1) x)], no pi,
 * order [x,y,z, sin(2^0 x),sin(2^0 y),sin(2^0 z), cos(2^0 x),cos(2^0 y),cos(2^0 z), ...] */
void r360o_pe(const double x[3], int32_t L, double* out) {
  int n = 0;
  for (int a = 0; a < 3; ++a) out[n++] = x[a];
  double f = 1.0;
  for (int l = 0; l < L; ++l) {
    for (int a = 0; a < 3; ++a) out[n++] = sin(f * x[a]);
    for (int a = 0; a < 3; ++a) out[n++] = cos(f * x[a]);
    f *= 2.0;
  }
}

/* y = W x + b, sums in index order, bias last (F) */
static void linear(const float* Wm, const float* b, int n_out, int n_in, const double* x, double* y) {
  for (int o = 0; o < n_out; ++o) {
    double acc = 0.0;
    for (int i = 0; i < n_in; ++i) acc += (double)Wm[(int64_t)o * n_in + i] * x[i];
    y[o] = acc + (double)b[o];
  }
}

#define MAX_W 512

/* Eq.1 with the tiny-MLP layout A1; raw = before head activations */
void r360o_field_raw(const r360o_scene* s, int32_t k, const float p[3], const float d[3], double out[4]) {
  const r360o_desc* D = &s->d;
  int Wd = D->hidden_width, pp = pe_dim(D->pe_pos_levels), pd = pe_dim(D->pe_dir_levels);
  double q[3], dd[3];
  for (int a = 0; a < 3; ++a) {                          /* A3, binary32 */
    float diff = p[a] - s->centre[(int64_t)k * 3 + a];
    float qa = diff * s->inv_half[(int64_t)k * 3 + a];
    q[a] = (double)qa;
    dd[a] = (double)d[a];
  }
  double x[MAX_W], y[MAX_W], in5[MAX_W];
  r360o_pe(q, D->pe_pos_levels, x);
  const float* w = s->w + (int64_t)k * s->P;
  int n_in = pp;
  for (int l = 0; l < D->n_hidden; ++l) {                /* trunk, ReLU */
    linear(w, w + (int64_t)Wd * n_in, Wd, n_in, x, y);
    w += (int64_t)Wd * n_in + Wd;
    for (int o = 0; o < Wd; ++o) x[o] = y[o] > 0.0 ? y[o] : 0.0;
    n_in = Wd;
  }
  double sigma_raw;
  linear(w, w + Wd, 1, Wd, x, &sigma_raw);               /* density head */
  w += Wd + 1;
  linear(w, w + (int64_t)Wd * Wd, Wd, Wd, x, in5);       /* feature, no activation (:439) */
  w += (int64_t)Wd * Wd + Wd;
  r360o_pe(dd, D->pe_dir_levels, in5 + Wd);              /* [feature, F(d)] */
  linear(w, w + (int64_t)Wd * (Wd + pd), Wd, Wd + pd, in5, y);
  w += (int64_t)Wd * (Wd + pd) + Wd;
  for (int o = 0; o < Wd; ++o) x[o] = y[o] > 0.0 ? y[o] : 0.0;   /* colour layer ReLU (:441) */
  double c[3];
  linear(w, w + 3 * Wd, 3, Wd, x, c);
  out[0] = sigma_raw; out[1] = c[0]; out[2] = c[1]; out[3] = c[2];
}

/* A4: sigma = softplus or ReLU (Table 4 :438); rgb = sigmoid (:442) */
void r360o_field(const r360o_scene* s, int32_t k, const float p[3], const float d[3], double out[4]) {
  double raw[4];
  r360o_field_raw(s, k, p, d, raw);
  if (s->d.density_activation == 1) out[0] = raw[0] > 20.0 ? raw[0] : log1p(exp(raw[0]));
  else out[0] = raw[0] > 0.0 ? raw[0] : 0.0;
  for (int c = 1; c < 4; ++c) out[c] = 1.0 / (1.0 + exp(-raw[c]));
}

/* ---------------------------------------------------------------- compositing (E, G)
 * Eq.4: C = sum w_i c_i, D = sum w_i t_i;
 * Eq.5 (:96-99): w_i = exp(-sum_{k<i} sigma_k delta_k) (1 - exp(-sigma_i delta_i));
 * reading E: delta_i = the stratum of sample i; reading G: running product,
 * stop after the first sample that makes T < tau. */
void r360o_composite(int64_t n, const double* sigma, const double* rgb, const float* t,
                     const float* delta, double tau, double out[6], double out_full[6], double* ambiguity) {
  double T = 1.0, C[3] = {0, 0, 0}, Dp = 0.0;
  double amb = INFINITY;
  int stopped = 0;
  for (int64_t i = 0; i < n; ++i) {
    double alpha = 1.0 - exp(-sigma[i] * (double)delta[i]);
    double w = T * alpha;
    for (int c = 0; c < 3; ++c) C[c] += w * rgb[i * 3 + c];
    Dp += w * (double)t[i];
    T = T * (1.0 - alpha);
    double m = fabs(T - tau) / tau;
    if (m < amb) amb = m;
    if (!stopped && T < tau) {
      stopped = 1;
      if (out) { out[0] = C[0]; out[1] = C[1]; out[2] = C[2]; out[3] = Dp; out[4] = T; out[5] = (double)(i + 1); }
    }
  }
  if (!stopped && out) { out[0] = C[0]; out[1] = C[1]; out[2] = C[2]; out[3] = Dp; out[4] = T; out[5] = (double)n; }
  if (out_full) { out_full[0] = C[0]; out_full[1] = C[1]; out_full[2] = C[2]; out_full[3] = Dp; out_full[4] = T; out_full[5] = (double)n; }
  if (ambiguity) *ambiguity = amb;
}

/* ---------------------------------------------------------------- render */

typedef struct {
  const r360o_scene* s;
  const float *o, *d;
  double T, C[3], Dp, amb;
  double Cs[3], Ds;    /* snapshot at the early-out sample */
  int stopped;
  uint32_t n_emitted, n_used;
} render_t;

static void render_visit(void* vctx, int64_t v, float t_in, float t_out, int occupied) {
  render_t* c = (render_t*)vctx;
  if (!occupied) return;
  const r360o_scene* s = c->s;
  int K = s->d.samples_per_voxel;
  double tau = (double)s->d.t_threshold;
  float len = t_out - t_in;
  float delta = len / (float)K;                                   /* D */
  int32_t k = s->label[v];                                         /* a4: voxel label */
  for (int j = 0; j < K; ++j) {
    float t = fmaf((float)j + 0.5f, delta, t_in);
    float p[3];
    for (int a = 0; a < 3; ++a) p[a] = fmaf(t, c->d[a], c->o[a]);
    double f[4];
    r360o_field(s, k, p, c->d, f);
    double alpha = 1.0 - exp(-f[0] * (double)delta);               /* G */
    double w = c->T * alpha;
    for (int ch = 0; ch < 3; ++ch) c->C[ch] += w * f[1 + ch];
    c->Dp += w * (double)t;
    c->T = c->T * (1.0 - alpha);
    c->n_emitted++;
    double m = fabs(c->T - tau) / tau;
    if (m < c->amb) c->amb = m;
    if (!c->stopped && c->T < tau) {
      c->stopped = 1;
      c->n_used = c->n_emitted;
      for (int ch = 0; ch < 3; ++ch) c->Cs[ch] = c->C[ch];
      c->Ds = c->Dp;
    }
  }
}

static void render_pixel(const r360o_scene* s, const float pose[12], const float* tab, int32_t W, int32_t H,
                         int i, int j, int64_t slot,
                         float* rgb, float* depth, float* rgb_full, float* depth_full,
                         float* ambiguity, uint32_t* n_emitted, uint32_t* n_used) {
  float o[3] = {pose[3], pose[7], pose[11]}, d[3];
  camera_dir(s, pose, tab, W, H, i, j, d);
  ray_t r;
  ray_setup(&r, o, d);
  render_t c;
  memset(&c, 0, sizeof(c));
  c.s = s; c.o = o; c.d = d; c.T = 1.0; c.amb = INFINITY;
  walk(s, &r, render_visit, &c);
  if (!c.stopped) {
    c.n_used = c.n_emitted;
    for (int ch = 0; ch < 3; ++ch) c.Cs[ch] = c.C[ch];
    c.Ds = c.Dp;
  }
  if (rgb) for (int ch = 0; ch < 3; ++ch) rgb[slot * 3 + ch] = (float)c.Cs[ch];
  if (depth) depth[slot] = (float)c.Ds;
  if (rgb_full) for (int ch = 0; ch < 3; ++ch) rgb_full[slot * 3 + ch] = (float)c.C[ch];
  if (depth_full) depth_full[slot] = (float)c.Dp;
  if (ambiguity) ambiguity[slot] = (float)c.amb;
  if (n_emitted) n_emitted[slot] = c.n_emitted;
  if (n_used) n_used[slot] = c.n_used;
}

int r360o_render_pixels(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                        int64_t n_pix, const int32_t* px, const int32_t* py,
                        float* rgb, float* depth, float* rgb_full, float* depth_full,
                        float* ambiguity, uint32_t* n_emitted, uint32_t* n_used) {
  if (!s || !pose || W < 1 || H < 1 || n_pix < 0) return 1;
  if (!r360o_pose_ok(pose)) return 1;                        /* B5 */
  float* tab = camera_tables(s, W, H);
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t q = 0; q < n_pix; ++q) {
    int i = px[q], j = py[q];
    if (i < 0 || i >= W || j < 0 || j >= H) { bad = 1; continue; }
    render_pixel(s, pose, tab, W, H, i, j, q, rgb, depth, rgb_full, depth_full, ambiguity, n_emitted, n_used);
  }
  free(tab);
  return bad;
}

int r360o_render_rows(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                      int32_t row0, int32_t row1,
                      float* rgb, float* depth, float* rgb_full, float* depth_full,
                      float* ambiguity, uint32_t* n_emitted, uint32_t* n_used) {
  if (!s || !pose || W < 1 || H < 1 || row0 < 0 || row1 > H || row0 > row1) return 1;
  if (!r360o_pose_ok(pose)) return 1;                        /* B5 */
  float* tab = camera_tables(s, W, H);
  int64_t n_pix = (int64_t)(row1 - row0) * W;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t q = 0; q < n_pix; ++q) {
    int i = (int)(q % W), j = row0 + (int)(q / W);
    render_pixel(s, pose, tab, W, H, i, j, q, rgb, depth, rgb_full, depth_full, ambiguity, n_emitted, n_used);
  }
  free(tab);
  return 0;
}

/* Bulk form of r360o_ray_samples for image rows [row0,row1): counts[ray] always; when t/subfield
 * are given they receive the samples ray-major at the exclusive prefix sum of counts (cap = their
 * length).  Returns the total number of samples, or -1 if it exceeds cap. */
int64_t r360o_samples_rows(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                           int32_t row0, int32_t row1, uint32_t* counts, int64_t cap, float* t,
                           int32_t* subfield) {
  if (!r360o_pose_ok(pose)) return -2;                       /* B5 */
  int64_t n_pix = (int64_t)(row1 - row0) * W;
  float* tab = camera_tables(s, W, H);
  float o[3] = {pose[3], pose[7], pose[11]};
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t q = 0; q < n_pix; ++q) {
    float d[3];
    camera_dir(s, pose, tab, W, H, (int)(q % W), row0 + (int)(q / W), d);
    counts[q] = (uint32_t)ray_samples(s, o, d, 0, NULL, NULL, NULL);
  }
  int64_t total = 0;
  for (int64_t q = 0; q < n_pix; ++q) total += counts[q];
  if (t && subfield) {
    if (total > cap) { free(tab); return -1; }
    int64_t* off = (int64_t*)malloc((size_t)(n_pix + 1) * sizeof(int64_t));
    off[0] = 0;
    for (int64_t q = 0; q < n_pix; ++q) off[q + 1] = off[q] + counts[q];
    float* dl = (float*)malloc((size_t)(total + 1) * sizeof(float));
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t q = 0; q < n_pix; ++q) {
      float d[3];
      camera_dir(s, pose, tab, W, H, (int)(q % W), row0 + (int)(q / W), d);
      ray_samples(s, o, d, counts[q], t + off[q], dl + off[q], subfield + off[q]);
    }
    free(dl);
    free(off);
  }
  free(tab);
  return total;
}

int r360o_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
