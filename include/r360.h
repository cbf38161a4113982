/* r360 -- B200-native equirectangular renderer for a radiance field made of
 * thousands of tiny local MLPs (the render hot path of 360Roam, arxiv 2208.02705).
 *
 * C ABI of libr360.so.  Citations are line numbers of the paper text
 * and readings listed in DESIGN.md.
 *
 * Problem statement (section 5.0.1): given the occupancy map, the
 * label of every occupied voxel ("each occupied voxel ... labeled to the
 * corresponding tiny MLP M_k") and the n tiny MLPs, render a 360-degree colour and
 * depth image for a camera pose by ray casting over occupied voxels, querying the
 * MLP that owns each sample, and volume rendering (Eq. 4-5).
 *
 * Conventions
 *  - "host" pointers are ordinary CPU memory, read during the call and never kept.
 *  - "device" pointers are CUDA device memory of the current device (for example
 *    torch.empty(..., device="cuda").data_ptr()), owned by the caller, written
 *    in stream order on the stream set with r360_set_stream (default: stream 0).
 *  - Every entry point returns a status; no exception or abort crosses the ABI.
 *    On failure outputs are unspecified and *out handles are NULL.
 *  - A handle may be used from one host thread at a time.
 *  - r360_render, r360_render_batch and r360_render_rows are ASYNCHRONOUS: they enqueue the frame on the
 *    scene's stream and return.  The buffers that hold a frame's samples are sized from the largest
 *    samples-per-ray ratio of earlier frames plus a quarter.  If a frame turns out to need more (a view with
 *    over 25 % more samples per ray than any before), the kernels of the affected ray chunk do nothing and the
 *    next call on the scene (r360_wait, r360_get_stats, any render or set call) renders that chunk again with
 *    larger buffers, in stream order: nothing is ever truncated.  So:
 *      - a caller that consumes the outputs through further r360 calls or after r360_get_stats needs nothing;
 *      - a caller that consumes them in its own stream work calls r360_wait(scene) first.  It waits until the
 *        frame's samples have been COUNTED (the first ~15 % of a frame), not for the frame, and returns
 *        immediately in the common case;
 *    The first frame a scene renders is sized from its exact count and waits for the GPU once per ray chunk.
 */
#ifndef R360_H
#define R360_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct r360_scene r360_scene; /* opaque; owns all device memory of a scene */

typedef enum {
  R360_OK = 0,
  R360_ERR_INVALID_ARG = 1, /* NULL pointer, non-positive size, unsupported width, non-finite pose ... */
  R360_ERR_BAD_LABEL = 2,   /* an occupied voxel whose subfield label is outside [0, n_subfields)   */
  R360_ERR_NONFINITE = 3,   /* NaN/Inf in the weights                                              */
  R360_ERR_CUDA = 4,        /* a CUDA call failed; r360_last_cuda_error() names it                 */
  R360_ERR_OOM = 5,         /* device (or host) allocation failed                                  */
  R360_ERR_CAPACITY = 6     /* a buffer provided by the caller (debug taps) is too small           */
} r360_status;

/* Scene description.  Geometry: DESIGN.md readings C (grid planes
 * P_a(k) = box_min_a + k * (box_max_a - box_min_a)/dims_a, binary32).
 * Network: readings A1-A4 ("6212 parameters"; Table 4 :434-444). */
/* Layout of the image outputs of the render calls (r360_set_output_format). */
typedef enum {
  R360_OUT_F32 = 0,      /* out_rgb float[.][3], out_depth float[.]  (default)                              */
  R360_OUT_RGB8_D16 = 1  /* out_rgb uint8[.][3] = round(255 * clamp(C, 0, 1)), out_depth IEEE binary16[.]:   */
                         /* 5 bytes per pixel instead of 16 for images that leave the GPU                   */
} r360_output_format;

typedef struct {
  int32_t dims[3];            /* Nx,Ny,Nz >= 1; linear voxel index = (iz*Ny+iy)*Nx+ix             */
  float box_min[3];           /* metres; box_max > box_min per axis (voxels may be anisotropic)    */
  float box_max[3];
  int32_t n_subfields;        /* n in [1, 65280]                                                   */
  int32_t hidden_width;       /* Wd: 32 or 64                                                      */
  int32_t n_hidden;           /* Hd in [1,8]: trunk layers before the density/feature layer        */
  int32_t pe_pos_levels;      /* L of F(p): 10 (63 inputs); [0,16] accepted                        */
  int32_t pe_dir_levels;      /* L of F(d): 4 (27 inputs); [0,8] accepted                          */
  int32_t samples_per_voxel;  /* K in [1,128]: stratum midpoints per occupied voxel crossed        */
  float t_threshold;          /* tau >= 0: stop a ray after the first sample with T < tau          */
  int32_t density_activation; /* 0 = ReLU (Table 4), 1 = softplus                    */
  uint8_t occ_threshold;      /* voxel occupied iff occupancy[i] >= occ_threshold (>= 1)           */
} r360_scene_desc;

/* Parameters per subfield for a description (6212 for Wd=32,Hd=2,L=10/4); 0 if invalid. */
int64_t r360_params_per_subfield(const r360_scene_desc* desc);

/* Create a scene.  All three arrays are HOST pointers and are copied.
 *  occupancy      uint8[N]  N = Nx*Ny*Nz, quantised occupancy probability
 *  voxel_subfield int32[N]  label in [0,n) of every occupied voxel; ignored where empty
 *  weights        float[n*P] per subfield, each layer W[out][in] row-major then b[out], in
 *                 the order trunk-1 (Wd x (3+6Lp)), trunk-2..Hd (Wd x Wd), density (1 x Wd),
 *                 feature (Wd x Wd), colour (Wd x (Wd+3+6Ld), input [feature, F(d)]), rgb (3 x Wd)
 * Errors: INVALID_ARG (NULL, dims < 1, box_max <= box_min, n out of range, Wd not 32/64, K out of
 * range, tau < 0 or NaN, occ_threshold 0), BAD_LABEL, NONFINITE, OOM, CUDA. */
r360_status r360_scene_create(const r360_scene_desc* desc, const uint8_t* occupancy,
                              const int32_t* voxel_subfield, const float* weights, r360_scene** out);

/* Free a scene and all its device memory.  NULL is a no-op. */
void r360_scene_destroy(r360_scene* scene);

/* Render one W x H view with the scene's camera (r360_set_camera; default: the equirectangular panorama of
 * Eq. 2-3) -- Eq. 2-5; steps a1-a10 of DESIGN.md.
 *  pose       HOST float[12]: row-major 3x4 [R|o], camera (x right, y down, z forward,
 *             PAPER.md:84) -> world; o = camera centre.  Must be finite, and R must not be (nearly) singular:
 *             2^-16 <= ||R||_F <= 2^16 and |det R| >= 2^-16 ||R||_F^3, evaluated in binary64 (DESIGN.md reading
 *             B5).  Every rotation passes, with or without a moderate scale; a matrix that maps some unit
 *             direction of Eq. 3 to (nearly) zero does not.  The same rule holds for every pose argument of
 *             this header (batches, graph poses, the fusion calls, the debug taps).
 *  out_rgb    DEVICE float[H*W*3], row-major, black background   (R360_OUT_RGB8_D16: uint8[H*W*3])
 *  out_depth  DEVICE float[H*W], Eq. 4's sum w_i t_i (radial distance; not opacity-normalised)
 *             (R360_OUT_RGB8_D16: binary16[H*W])
 * Asynchronous (see "Conventions").  Errors: INVALID_ARG (NULL, W < 1, H < 1, non-finite or singular pose), OOM, CUDA;
 * CAPACITY inside a CUDA stream capture when a buffer would have to be allocated (see r360_graph_status). */
r360_status r360_render(r360_scene* scene, const float pose[12], int32_t W, int32_t H,
                        void* out_rgb, void* out_depth);

/* Same for B poses (HOST float[B*12]); outputs DEVICE [B*H*W*3], [B*H*W].  The poses of a batch are binned
 * together, so a subfield's weights are staged once for all of them: a stereoscopic pair (PAPER.md:172-174,
 * Fig. 5: "monoscopic ... and stereoscopic modes") is a batch of two poses one eye distance apart. */
r360_status r360_render_batch(r360_scene* scene, const float* poses, int32_t B, int32_t W, int32_t H,
                              void* out_rgb, void* out_depth);

/* A band of image rows [row0, row1) of one view: rays are independent ("each ray can be concurrently processed",
 * PAPER.md:174), so a frame splits across GPUs by rows with no exchange but the gather of the bands (SURVEY.md
 * 8(e)).  out_rgb / out_depth point at the BAND: DEVICE [(row1-row0)*W*3], [(row1-row0)*W]; pass
 * frame + row0*W*3 (and frame_depth + row0*W) to render into a full-size frame in place.  The pixels are
 * bit-identical to the same rows of r360_render.  INVALID_ARG unless 0 <= row0 < row1 <= H. */
r360_status r360_render_rows(r360_scene* scene, const float pose[12], int32_t W, int32_t H, int32_t row0,
                             int32_t row1, void* out_rgb, void* out_depth);

/* End-to-end call: like r360_render_batch but the outputs are HOST buffers ([B*H*W*3], [B*H*W] in the
 * scene's output format; pinned memory for full PCIe speed).  Every chunk of rays (r360_set_chunk_rays; a call
 * that fits one chunk can be cut into bands, r360_set_host_bands) is copied device -> host on a second
 * stream while the next chunk is rendered; the call returns when all copies are done, also after an error. */
r360_status r360_render_batch_host(r360_scene* scene, const float* poses, int32_t B, int32_t W, int32_t H,
                                   void* out_rgb_host, void* out_depth_host);
/* A call that fits one ray chunk can be cut into `bands` (1..64) chunks so that a band's copy runs behind the next
 * band's kernels.  Default 1: measured on config 3 (2048 x 1024), every extra chunk costs 0.13 ms of kernel tails,
 * more than the copy it hides. */
r360_status r360_set_host_bands(r360_scene* scene, int32_t bands);

/* Streaming form of r360_render_batch_host: returns when the frame and its copy to the host are enqueued.  Two
 * staging buffers are used in turn, so the copy of one frame runs behind the kernels of the next: a stream of
 * frames costs max(render, copy) per frame instead of their sum.  The host buffers of a call must stay valid, and
 * hold the frame, once r360_host_sync (or the second-next r360_render_batch_host_async) has returned. */
r360_status r360_render_batch_host_async(r360_scene* scene, const float* poses, int32_t B, int32_t W, int32_t H,
                                         void* out_rgb_host, void* out_depth_host);
/* Waits until every frame enqueued by r360_render_batch_host_async is in its host buffers. */
r360_status r360_host_sync(r360_scene* scene);

/* Returns once the outputs of the last render call are guaranteed complete IN STREAM ORDER (see "Conventions"):
 * waits for the frame's sample count, re-renders a chunk whose samples exceeded the buffers.  Does not wait for
 * the frame itself.  Also returns the status of such a re-render (OOM, CUDA). */
r360_status r360_wait(r360_scene* scene);

/* Image output layout of the following render calls (r360_output_format).  INVALID_ARG for another value. */
r360_status r360_set_output_format(r360_scene* scene, int32_t format);

/* Pre-size the sample buffers for chunks of up to max_rays_per_chunk rays with segments_per_ray occupied voxels
 * crossed per ray on average (x 1.25), so that no later frame has to grow them. */
r360_status r360_reserve(r360_scene* scene, uint64_t max_rays_per_chunk, double segments_per_ray);

/* CUDA graphs.  The render calls may be captured (cudaStreamBeginCapture on the scene's stream) once the scene
 * has rendered a frame of the same size outside a capture (which builds the pixel tables and sizes the buffers;
 * a capture that would have to allocate returns R360_ERR_CAPACITY).  The captured frame reads its poses from a
 * pinned buffer of the scene at every replay: r360_set_graph_poses replaces them between replays (host memcpy,
 * no CUDA call).  A replay cannot re-render a chunk that outgrew the buffers: r360_graph_status synchronises the
 * stream and returns R360_ERR_CAPACITY if the last replay hit that case (its outputs are then incomplete; call
 * r360_reserve with a larger ratio and capture again), R360_OK otherwise.
 * A graph holds the ADDRESSES and capacities of the scene's buffers as they were at capture.  Any later call outside
 * a capture that frees or reallocates one of them makes the graph STALE, and a replay would touch freed memory: a
 * larger frame or chunk, another image size or camera (new pixel tables), more poses per batch, a chunk that had to be
 * re-rendered with larger buffers, r360_reserve, a switch to the tensor path or to wavefront passes for the first
 * time.  The scene counts these events: for a stale graph r360_graph_status and r360_set_graph_poses return
 * R360_ERR_CAPACITY -- check one of them before every replay that follows other calls on the scene, and capture again.
 * Call r360_wait before cudaStreamBeginCapture: a captured render call returns R360_ERR_INVALID_ARG while chunks of the
 * previous frame are still unverified (inside a capture they could not be re-rendered and would be lost). */
r360_status r360_set_graph_poses(r360_scene* scene, const float* poses, int32_t B);
r360_status r360_graph_status(r360_scene* scene);

/* Algorithm 1, stage II (text :157): geometry-aware assignment of the occupied voxels to
 * n tiny networks -- "pop an unassigned voxel with the minimum coordinate as the anchor; search s-1 nearest
 * unassigned neighbours; assign these s voxels to the k-th network", s = S/n.  Readings (S1-S4): the
 * first S mod n networks take one voxel more; minimum coordinate = smallest linear index; nearest = squared
 * distance of voxel centres in metres (binary32, each operation rounded); ties to the smaller linear index.
 * Runs on the current CUDA device.  dims/box as in r360_scene_desc; occupancy: HOST uint8[N], occupied iff
 * >= occ_threshold (>= 1); labels_out: HOST int32[N], receives the network of every occupied voxel and -1 for
 * empty ones -- the voxel_subfield input of r360_scene_create.  Caller owns both arrays.
 * R360_ERR_INVALID_ARG: null pointers, bad dims/box, n < 1, n > S, dims > 65535, S >= 2^25. */
r360_status r360_assign_subfields(const int32_t dims[3], const float box_min[3], const float box_max[3],
                                  const uint8_t* occupancy, uint8_t occ_threshold, int32_t n,
                                  int32_t* labels_out);

/* Floorplan estimation from the occupancy map (section 5.0.2; Fig. 6): the occupied voxels of
 * the upper slice (default 60-65 % of the height) are projected to the floor plane, closed by a 3x3 square
 * ("simple morphological operations"), the free region around the seed cell is segmented out with its inner
 * boundary, and the occupied voxels of the lower slice (default 20-30 %) inside it are added as obstacles.
 * Readings F1-F7 in DESIGN.md (height axis = z; a layer belongs to a slice iff its centre fraction lies in it;
 * 4-connectivity).  Runs on the current CUDA device.  occupancy: HOST uint8[N] as in r360_scene_create;
 * (seed_x, seed_y): a free cell inside the region to map (the viewer's position); upper / lower: {lo, hi}
 * fractions of the height, or NULL for the paper's values; plan_out: HOST uint8[Ny*Nx], bit 0 interior, bit 1
 * inner boundary, bit 2 obstacle (the floorplan of Fig. 6c = bits 1|2).  Caller owns all arrays.
 * R360_ERR_INVALID_ARG: null pointers, bad dims, seed outside the image or on a wall cell, lo > hi. */
r360_status r360_floorplan(const int32_t dims[3], const uint8_t* occupancy, uint8_t occ_threshold,
                           int32_t seed_x, int32_t seed_y, const float upper[2], const float lower[2],
                           uint8_t* plan_out);

/* Progressive probabilistic occupancy, one observation (Eq. 6; Algorithm 1 stage I): a depth
 * panorama (Eq. 4's radial distance) and optionally an uncertainty panorama seen from `pose` are fused into the
 * log-odds grid, logit(p|z_1:t) = logit(p|z_1:t-1) + logit(p|z_t), clamped to [-2, 3.5] (:119-122).  Readings
 * O1-O5 in DESIGN.md: Octomap's scan insertion and defaults (the framework the paper adopts; its default clamps
 * are the paper's): a voxel holding the end point of a ray gets + ln(p/(1-p)), p = 0.5 + 0.2 (1 - u), u the smallest
 * uncertainty in [0,1] of the rays ending there (0 without a map); a voxel only crossed before the end points gets
 * ln(0.4/0.6); pixels with depth <= 0 or non-finite are skipped; a voxel is occupied iff logit > ln(0.97/0.03).
 * Runs on the current CUDA device.  logodds: HOST float[N], read and written; pose: HOST float[12] as in
 * r360_render; depth, uncertainty (may be NULL): HOST float[H*W] of a W x H equirectangular image.
 * R360_ERR_INVALID_ARG: null pointers, bad dims/box, W or H < 1, non-finite pose. */
r360_status r360_occupancy_fuse(const int32_t dims[3], const float box_min[3], const float box_max[3],
                                float* logodds, const float pose[12], int32_t W, int32_t H,
                                const float* depth, const float* uncertainty);

/* The same with the log-odds grid RESIDENT ON THE DEVICE between observations (Algorithm 1 stage I fuses the
 * panoramas progressively): create once (logodds_init: HOST float[N] or NULL for zeros), fuse any
 * number of observations (r360_fusion_fuse: HOST depth / uncertainty images; r360_fusion_fuse_device: DEVICE images,
 * e.g. the depth output of r360_render), read back when needed (logodds_out: HOST float[N] or NULL; occupancy_out:
 * HOST uint8[N] or NULL, 255 where logit > ln(0.97/0.03), else 0 -- the occupancy input of r360_scene_create with
 * occ_threshold 128).  Work runs on the default (legacy) stream of the current device; r360_fusion_read synchronises.
 * Feeding r360_fusion_fuse_device from r360_render: the render calls are asynchronous and run on the scene's stream,
 * so (1) call r360_wait(scene) first -- a chunk that outgrew its buffers is only complete after that -- and (2) if the
 * scene's stream does not synchronise with the legacy default stream (a cudaStreamNonBlocking stream, or a process
 * built with per-thread default streams), order the two yourself: cudaStreamSynchronize(scene stream), or an event
 * recorded there and waited for on stream 0, before r360_fusion_fuse_device.  With the scene on stream 0 (the
 * default) or on an ordinary blocking stream, r360_wait alone is enough. */
typedef struct r360_fusion r360_fusion;
r360_status r360_fusion_create(const int32_t dims[3], const float box_min[3], const float box_max[3],
                               const float* logodds_init, r360_fusion** out);
r360_status r360_fusion_fuse(r360_fusion* fusion, const float pose[12], int32_t W, int32_t H, const float* depth,
                             const float* uncertainty);
r360_status r360_fusion_fuse_device(r360_fusion* fusion, const float pose[12], int32_t W, int32_t H,
                                    const float* depth, const float* uncertainty);
r360_status r360_fusion_read(r360_fusion* fusion, float* logodds_out, uint8_t* occupancy_out);
void r360_fusion_destroy(r360_fusion* fusion);

/* One observation of Eq. 6 WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc:
 * a program whose own arena or caching allocator already holds the whole GPU (a library allocation would fail or
 * fragment it), a frame loop that cannot afford the device-wide stall cudaMalloc / cudaFree may cause, or code that
 * runs at a moment when its process forbids allocation (e.g. another thread is recording a CUDA graph in the global
 * capture mode).  r360_fusion_create / r360_fusion_fuse* allocate (grid-sized scratch at create, tables and staging
 * whenever the image size changes); this call uses neither cudaMalloc nor cudaFree nor any allocating library
 * routine.  Same arithmetic and same kernels as r360_fusion_fuse_device: the grid is equal bit for bit.
 *  dims, box_min, box_max  HOST, as in r360_fusion_create
 *  logodds      DEVICE float[N], N = Nx*Ny*Nz, read and written in place (the caller's grid; this call keeps no state)
 *  pose         HOST float[12] as in r360_render; read before the call returns
 *  depth        DEVICE float[H*W];  uncertainty  DEVICE float[H*W] or NULL
 *  cuda_stream  cudaStream_t as void* (NULL = the default stream); all work is enqueued on it, the call does not wait
 * Scratch: the per-voxel flags and minimum uncertainty (8 bytes per voxel), the pixel-angle tables and the pose live
 * in one static device array of 64 MiB + 48 KiB inside libr360.so.  Every GPU that loads the library holds it until
 * the process exits, and it bounds the problem: N <= R360_STATIC_MAX_VOXELS, W <= R360_STATIC_MAX_W,
 * H <= R360_STATIC_MAX_H; anything larger returns R360_ERR_CAPACITY before any GPU work (r360_last_cuda_error() then
 * names the limits) -- use the r360_fusion handle for such grids.
 * The FIRST call on each device looks up the array's device address (once, with that device current) and may make
 * the CUDA runtime load the library's kernels: make that first call during set-up, before any stream capture.
 * Every call on a device shares the one array and leaves its last contents there; a call resets the part it uses
 * before its kernels run.  Calls whose GPU work can overlap (two streams, two host threads with their own streams)
 * race on it: keep all calls of a device on one stream, or order them with events.
 * Errors: INVALID_ARG (NULL pointers, dims < 1, box_max <= box_min, W or H < 1, non-finite pose, device ordinal
 * >= 64), CAPACITY (see above), CUDA. */
#define R360_STATIC_MAX_VOXELS (8u << 20) /* 8 Mi voxels: covers 256 x 256 x 96 (BASELINE configs 1-3, 5)     */
#define R360_STATIC_MAX_W 4096
#define R360_STATIC_MAX_H 2048
r360_status r360_fusion_fuse_static(const int32_t dims[3], const float box_min[3], const float box_max[3],
                                    float* logodds, const float pose[12], int32_t W, int32_t H, const float* depth,
                                    const float* uncertainty, void* cuda_stream);

/* Camera of the following render / debug calls.  model 0 (default) = the equirectangular panorama of
 * Eq.2-3; model 1 = pinhole view for roaming (the paper's perspective display,
 * PAPER.md:206, :200, gives no model; reading P): pixel centre (i+0.5, j+0.5) ->
 * x = (i + 0.5 - cx)/fx, y = (j + 0.5 - cy)/fy (binary64, rounded once to binary32),
 * d_cam = (x, y, 1)/|(x, y, 1)| in the camera frame of Eq.3 (x right, y down, z forward), d = R d_cam;
 * depth stays the distance along the unit ray.  fx, fy, cx, cy in pixels; fx, fy > 0; ignored for model 0.
 * Returns R360_ERR_INVALID_ARG for another model or non-finite / non-positive intrinsics. */
r360_status r360_set_camera(r360_scene* scene, int32_t model, double fx, double fy, double cx, double cy);

/* Wavefronted early termination: mode 0 = off (default), 1 = on, 2 = automatic.  On: the occupied voxels a ray
 * crosses are fed to the MLP in passes (crossings [0,2), [2,6), [6,16), [16,64), [64,inf) of every ray); after each
 * pass the compositing step retires the rays whose transmittance fell below t_threshold (Eq.4-5, reading G), so
 * their remaining samples are never evaluated.  The images are the same as with 0 (same per-ray sequence of
 * operations).  It pays when surfaces are opaque, as in trained scenes (config 5 made opaque: 8.2 -> 3.0 ms), and
 * costs about 0.6 ms of extra launches on a 2048 x 1024 frame when no ray terminates early.  Automatic: a frame is
 * rendered in passes iff the last finished frame of the scene composited less than half of its samples.
 * While passes are in use, r360_stats.segments / mlp_tiles count what reached the MLP, and the per-stage times cover
 * the first pass. */
r360_status r360_set_wavefront(r360_scene* scene, int32_t mode);

/* Arithmetic of the tiny MLPs (steps a6-a9; Eq.1, Table 4):
 *  0 = binary32 on the FP32 ALUs (default; within 1e-4 of the oracle);
 *  1 = tensor cores (tcgen05), operands (weights, positional encoding, activations) rounded to bfloat16,
 *      binary32 accumulation -- BASELINE.json's "bf16 tensor-core variant";
 *  2 = the same kernel with binary16 operands (11 significant bits instead of 8, same speed): THE tensor mode for scenes
 *      whose pixels are decided by one or two samples (opaque surfaces), where bfloat16's per-sample colour error
 *      (up to 2.4e-3, above the 2e-3 bar) is not averaged out; mode 2 stays within 5e-4 there.  Mode 1 is within
 *      2e-3 only where a pixel averages many samples (all five BASELINE.json scenes).  DESIGN.md section 6 has the
 *      per-layer error table.
 * R360_ERR_INVALID_ARG: unknown mode; modes 1-2 for a network the tensor kernel does not cover (positional
 * encodings other than L = 10 / 4, or weight buffers that exceed the SM's shared memory: Wd = 32 with more than 6
 * trunk layers, Wd = 64 with more than 3); mode 2 when a weight, a bias or a product of the folded feature and
 * colour layers exceeds binary16's range (65504). */
r360_status r360_set_precision(r360_scene* scene, int32_t mode);
/* CUDA stream (cudaStream_t / CUstream as void*) all work of this scene is enqueued on. */
r360_status r360_set_stream(r360_scene* scene, void* cuda_stream);
/* Upper bound on rays processed per internal chunk (default 4 Mi). */
r360_status r360_set_chunk_rays(r360_scene* scene, int64_t max_rays);

typedef struct {
  uint64_t rays;             /* of the last render call                                            */
  uint64_t segments;         /* occupied voxels crossed, summed over rays                          */
  uint64_t samples_emitted;  /* K * segments (geometric; bit-exact contract)                       */
  uint64_t samples_used;     /* samples composited before early-out (floating point; not exact)    */
  uint64_t mlp_tiles;        /* 128-row tiles the MLP kernel processed                             */
  uint32_t chunks;           /* ray chunks                                                         */
  uint32_t kernel_launches;  /* kernels of this library launched by the last render call           */
  float ms_count;            /* device time per stage of the last render call, CUDA events         */
  float ms_scan;
  float ms_emit;
  float ms_mlp;
  float ms_composite;
  float ms_total;
  uint32_t retries;          /* chunks rendered again because they outgrew the buffers, since scene creation */
} r360_stats;

/* Statistics of the last render call; synchronises the scene's stream (and settles the call like r360_wait). */
r360_status r360_get_stats(r360_scene* scene, r360_stats* out);

/* Debug tap for the parity tests (steps a1-a5): runs the sampler and the binning for
 * one pose and exports, ray-major (ray = j*W + i):
 *  counts  DEVICE uint32[W*H]   samples of each ray (K x occupied voxels crossed)
 *  offsets DEVICE uint32[W*H]   exclusive prefix sum of counts
 *  t       DEVICE float[cap]    sample distances, front to back per ray
 *  subfield DEVICE int32[cap]   owning subfield of each sample (read back from the bins)
 *  total   HOST uint64*         total samples; R360_ERR_CAPACITY if total > cap (t/subfield
 *                               untouched, counts/offsets/total valid) */
r360_status r360_debug_samples(r360_scene* scene, const float pose[12], int32_t W, int32_t H,
                               uint32_t* counts, uint32_t* offsets, float* t, int32_t* subfield,
                               uint64_t cap, uint64_t* total);

/* The same plus steps a6-a9: the tiny MLPs are evaluated (in the scene's precision mode) and
 *  field   DEVICE float[cap*4]  (sigma, r, g, b) of every sample, in the order of t / subfield
 * is exported before any compositing -- the parity tap for the field (Eq.1, Table 4) sample by sample. */
r360_status r360_debug_field(r360_scene* scene, const float pose[12], int32_t W, int32_t H,
                             uint32_t* counts, uint32_t* offsets, float* t, int32_t* subfield, float* field,
                             uint64_t cap, uint64_t* total);

const char* r360_status_string(r360_status s);
/* Text of the last CUDA error seen by this library on the calling thread ("" if none). */
const char* r360_last_cuda_error(void);
/* "r360 <version> sm_100a" */
const char* r360_version(void);

#ifdef __cplusplus
}
#endif
#endif
