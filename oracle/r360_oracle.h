/* r360 ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-purpose CPU restatement of the 360Roam render path
 * (arxiv 2208.02705; citations are /root/reference/PAPER.md line numbers).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, link or call anything in oracle/.
 * It shares no code, header, table or helper with paper_2208_02705_b200/
 * or include/; the two sides agree only through DESIGN.md and the paper.
 *
 * Precision: everything that decides an INTEGER (which voxels a ray crosses,
 * how many samples it gets, which subfield owns them) and every sample position
 * is computed in IEEE binary32 with individually rounded operations (compile
 * with -ffp-contract=off, no fast-math), because the CUDA path must reproduce
 * those bits.  The field evaluation (positional encoding, tiny MLP, heads) and
 * the compositing sums are evaluated in binary64 from those binary32 inputs and
 * the binary32 weights; results are rounded to binary32 once on output.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Eq.2/3 round trip and cardinal
 * directions; brute-force voxel predicate and dense marching for the walk;
 * parameter count 6212; one-hot PE probes; float64 PyTorch
 * re-evaluation of the MLP; slab / constant-colour / telescoping closed forms
 * for Eq.4-5; zero-weight end-to-end closed form.
 * Unpinned against the authors' system (not available): pi-free PE, per-subfield
 * normalisation, K, midpoints, tau, softplus, pixel centres -- DESIGN.md readings.
 */
#ifndef R360_ORACLE_H
#define R360_ORACLE_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t dims[3];        /* Nx,Ny,Nz ; linear voxel index = (iz*Ny+iy)*Nx+ix            */
  float box_min[3];
  float box_max[3];
  int32_t n_subfields;
  int32_t hidden_width;   /* Wd */
  int32_t n_hidden;       /* Hd: trunk layers before the density/feature layer          */
  int32_t pe_pos_levels;  /* L for position (10) */
  int32_t pe_dir_levels;  /* L for direction (4) */
  int32_t samples_per_voxel; /* K */
  float t_threshold;      /* tau */
  int32_t density_activation; /* 0 ReLU (Table 4), 1 softplus */
  int32_t occ_threshold;  /* occupied iff occupancy[i] >= occ_threshold */
} r360o_desc;

typedef struct r360o_scene r360o_scene;

/* Returns NULL on invalid arguments. Copies all inputs. */
r360o_scene* r360o_create(const r360o_desc* desc, const uint8_t* occupancy,
                          const int32_t* voxel_subfield, const float* weights);
void r360o_destroy(r360o_scene* s);
int64_t r360o_params_per_subfield(const r360o_desc* desc);

/* Eq.2 inverse at pixel centres (reading B1), tables rounded once to binary32 (B2). */
void r360o_trig_tables(int32_t W, int32_t H, float* sin_phi, float* cos_phi,
                       float* sin_theta, float* cos_theta);
/* Eq.2 forward: (phi,theta) -> (u,v), binary64. */
void r360o_sphere_to_pixel(double phi, double theta, int32_t W, int32_t H, double* u, double* v);
/* Pixel centre -> (phi,theta), binary64 (reading B1). */
void r360o_pixel_to_sphere(int32_t i, int32_t j, int32_t W, int32_t H, double* phi, double* theta);
/* Ray of pixel (i,j): o = pose translation, d = R * Eq.3 direction (binary32, B3). */
void r360o_ray(const float pose[12], int32_t W, int32_t H, int32_t i, int32_t j, float o[3], float d[3]);

/* Pinhole view (reading P; the paper's perspective display, gives no model):
 * x_i = (i + 0.5 - cx)/fx, y_j = (j + 0.5 - cy)/fy in binary64 rounded once to binary32;
 * d_cam = (x, y, 1)/|(x, y, 1)| in binary32 (n2 = (x*x + y*y) + 1, inv = 1/sqrt(n2)); d = R d_cam (B3). */
void r360o_pinhole_tables(int32_t W, int32_t H, double fx, double fy, double cx, double cy, float* x, float* y);
void r360o_ray_pinhole(const float pose[12], double fx, double fy, double cx, double cy, int32_t i, int32_t j,
                       float o[3], float d[3]);
/* Camera used by r360o_ray_samples / render_* / samples_rows of this scene: model 0 = equirectangular
 * (default), 1 = pinhole with the given intrinsics (pixels).  Returns 0 on success. */
int r360o_set_camera(r360o_scene* s, int32_t model, double fx, double fy, double cx, double cy);

/* Voxel walk (readings C1-C5).  Writes up to cap crossed voxels front to back;
 * only_occupied != 0 keeps occupied voxels only.  Returns the number found
 * (may exceed cap; then only cap were written). */
int64_t r360o_walk(const r360o_scene* s, const float o[3], const float d[3], int only_occupied,
                   int64_t cap, int32_t* voxel, float* t_in, float* t_out);
/* Box clip (C2): returns 1 and [t0,t1] if the ray has a non-empty interval. */
int r360o_clip(const r360o_scene* s, const float o[3], const float d[3], float* t0, float* t1);

/* Reading B5: 1 iff the pose is admissible (finite; 3x3 part M with 2^-16 <= |M|_F <= 2^16 and
 * |det M| >= 2^-16 |M|_F^3 in binary64).  The render / sample functions below return an error (1, or -2 where they
 * return a count) for any other pose. */
int r360o_pose_ok(const float pose[12]);
/* Samples of one pixel's ray (reading D). Returns count (may exceed cap). */
int64_t r360o_ray_samples(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                          int32_t i, int32_t j, int64_t cap, float* t, float* delta, int32_t* subfield);

/* Per-subfield normalisation (reading A3): centre and 1/half-extent, binary32. */
void r360o_subfield_frame(const r360o_scene* s, int32_t k, float centre[3], float inv_half[3]);
/* Positional encoding (A2) of a 3-vector, binary64, 3+6L outputs. */
void r360o_pe(const double x[3], int32_t L, double* out);
/* Field of subfield k at world point p, unit direction d: out = {sigma, r, g, b} (binary64). */
void r360o_field(const r360o_scene* s, int32_t k, const float p[3], const float d[3], double out[4]);
/* Raw network outputs before the heads' activations: {sigma_raw, r_raw, g_raw, b_raw}. */
void r360o_field_raw(const r360o_scene* s, int32_t k, const float p[3], const float d[3], double out[4]);

/* Eq.4-5 with per-sample stratum delta (reading E) and early-out (reading G).
 * out = {R,G,B,D,T_end, n_used}; out_full = same without early-out; *ambiguity =
 * min_i |T_i - tau| / tau over all samples (G4). Any output pointer may be NULL. */
void r360o_composite(int64_t n, const double* sigma, const double* rgb, const float* t,
                     const float* delta, double tau, double out[6], double out_full[6], double* ambiguity);

/* Render a list of pixels (px[i],py[i]).  Outputs (any may be NULL), per pixel:
 * rgb[3], depth, rgb_full[3]/depth_full (no early-out), ambiguity, n_emitted, n_used. */
int r360o_render_pixels(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                        int64_t n_pix, const int32_t* px, const int32_t* py,
                        float* rgb, float* depth, float* rgb_full, float* depth_full,
                        float* ambiguity, uint32_t* n_emitted, uint32_t* n_used);
/* Render image rows [row0,row1) (every pixel); outputs sized (row1-row0)*W. */
int r360o_render_rows(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                      int32_t row0, int32_t row1,
                      float* rgb, float* depth, float* rgb_full, float* depth_full,
                      float* ambiguity, uint32_t* n_emitted, uint32_t* n_used);
/* Bulk sample tap for rows [row0,row1): counts[(row1-row0)*W]; optional t/subfield (length cap),
 * ray-major at the exclusive prefix sum of counts.  Returns total samples, -1 if > cap. */
int64_t r360o_samples_rows(const r360o_scene* s, const float pose[12], int32_t W, int32_t H,
                           int32_t row0, int32_t row1, uint32_t* counts, int64_t cap, float* t,
                           int32_t* subfield);
int r360o_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
