/* sssgs.h -- C ABI of libsssgs: the forward relighting render path of SSS-GS
 * ("Subsurface Scattering for 3D Gaussian Splatting", arXiv 2408.12282) on one B200.
 *
 * Citations "L<n>" are line numbers of the paper text; "S<k>" are the readings
 * of points the paper leaves open, listed in DESIGN.md.
 *
 * The path (Fig. 2, L87-116):
 *   1. per Gaussian and per (view, light): the joint MLP
 *        (L_SSS, L_in) = f_Theta(mu, Sigma, n, w_in, w_out, v)            (Eq. 6; L347)
 *   2. EWA projection Sigma' = J W Sigma W^T J^T (Eq. 2), tile binning, depth sort,
 *      front-to-back alpha compositing C = sum_i prod_{j<i}(1-alpha_j) alpha_i c_i (Eq. 3,
 *      L68-72) of a 16-channel G-buffer (L55, L114)
 *   3. per-pixel deferred shading (L114): Cook-Torrance/GGX + diffuse (Eq. 4) times the
 *      learned incident light, blended with the SSS residual (Eq. 7).
 *
 * Conventions
 *   - Every pointer inside sssgs_gaussians / sssgs_mlp / sssgs_out is a DEVICE pointer for
 *     sssgs_render and a HOST pointer for sssgs_render_host.  cams / lights are HOST arrays.
 *     All cameras of one call must share one image size (frames are laid out [F][H][W]).
 *   - All memory reachable through the argument structs is caller-owned: the library never
 *     frees it and never keeps a pointer to it after the call's work has finished.
 *   - Device pointers must be 16-byte aligned; arrays are dense, row-major, fp32 unless noted.
 *   - Work is enqueued on the given CUDA stream; sssgs_render never synchronises and is
 *     CUDA-graph-capture safe.  Results are valid once the caller has synchronised the stream.
 *     Internally the MLP runs on a stream owned by the context, forked from and joined back to
 *     the caller's stream with events inside the same call (so it overlaps the geometry stages);
 *     to the caller the call behaves as if everything ran on the given stream.
 *   - Every function returns 0 (SSSGS_OK) or a negative sssgs_status; no exceptions or aborts
 *     cross the ABI.  sssgs_last_error() returns a human-readable description.
 *   - There is no CPU fallback: without an sm_100 device sssgs_create fails (SSSGS_EARCH).
 *   - A context belongs to the device of sssgs_config.device: every entry point makes that device
 *     current for the duration of the call and restores the caller's device before returning, so
 *     contexts on several GPUs can be driven from one thread.
 */
#ifndef SSSGS_H_
#define SSSGS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SSSGS_OK = 0,
  SSSGS_EINVAL = -1,    /* bad argument (NULL, dimension mismatch, misaligned pointer, ...)   */
  SSSGS_ECAPACITY = -2, /* a size exceeds what the context was created for                    */
  SSSGS_ECUDA = -3,     /* a CUDA runtime call failed                                         */
  SSSGS_EARCH = -4,     /* device is not compute capability 10.x                              */
  SSSGS_EOVERFLOW = -5  /* (sssgs_render_host only) tile-instance buffer overflowed           */
} sssgs_status;

enum { SSSGS_ACT_RELU = 0, SSSGS_ACT_LEAKY_RELU = 1 };
enum { SSSGS_F32 = 0, SSSGS_BF16 = 1 };
/* sssgs_mlp.compute: 16-bit type of the tensor-core operands (weights and every layer input) */
enum { SSSGS_COMPUTE_FP16 = 0, SSSGS_COMPUTE_BF16 = 1 };

/* flags of sssgs_render */
enum {
  SSSGS_LIGHTS_PER_CAMERA = 1u,/* lights is [n_cam][n_light] (camera c uses its own n_light
                                  lights) instead of one shared [n_light] list            */
  SSSGS_SUM_LIGHTS = 2u,       /* image-based lighting as a sum of point lights (PAPER.md L301,
                                  App. D): out.rgb holds ONE frame per camera, [n_cam][H][W][3] =
                                  sum over the call's lights of intensity_l * A * L_out,l, plus the
                                  background term (1 - A) bg once.  The sum is formed in the
                                  rasteriser's epilogue (no per-light frames are written).
                                  gbuffer / mlp_out stay per light; the AOVs must be NULL.    */
  SSSGS_TIGHT_LISTS = 8u,      /* tight tile lists (reading S5; "efficiently designed
                                  splatting technique"): a (tile, Gaussian) pair of the canonical list is
                                  kept only if the Gaussian's alpha >= 1/255 support box reaches a pixel of
                                  the tile.  The list is a sub-sequence of the canonical one (same order),
                                  contains every pair with alpha >= 1/255 at some pixel of the tile, and
                                  blends the same (pixel, entry) pairs: frames are bit-identical to the
                                  canonical list's on images of more than 1600 tiles, and equal up to the
                                  order of the per-slot partial sums (last bits) on smaller ones; sorted_keys /
                                  sorted_vals / tile_ranges / SSSGS_CNT_INSTANCES then describe the tight
                                  list.  ~0.6-0.75 x the instances: less to emit, sort and walk.        */
  SSSGS_FORWARD_SHADING = 4u,  /* the "w/o deferred" variant of the paper's ablation (PAPER.md L283
                                  Tab. 2, Fig. 5): Eq. 7 is evaluated per Gaussian (at its
                                  centre, with its own normal and material) and the RGB values are
                                  composited (Eq. 3): out.rgb = sum_i T_i alpha_i c_i + (1 - A) bg.
                                  gbuffer and the AOVs must be NULL; not combinable with
                                  SSSGS_SUM_LIGHTS.                                            */
  SSSGS_BACKWARD_FP32 = 16u    /* sssgs_render_backward only: run the MLP backward in fp32 on the CUDA
                                  cores instead of the tensor cores (slower; the reference path of the
                                  parity tests, and what MLPs with incident-head hidden layers use).  */
};

/* indices into sssgs_out.counters (int64 each, per camera: counters[cam*SSSGS_NCOUNTERS + k]) */
enum {
  SSSGS_CNT_NVIS = 0,      /* Gaussians that survive projection/culling                       */
  SSSGS_CNT_INSTANCES = 1, /* I = sum of tiles touched (tile list length, before clamping to
                              max_instances; saturates at 2^30 - 1, which always flags overflow) */
  SSSGS_CNT_OVERFLOW = 2,  /* 1 if I > max_instances: the frame content is then undefined    */
  SSSGS_CNT_SORT_ERROR = 3,/* non-zero if a look-back wait exceeded its spin bound (bug trap) */
  SSSGS_CNT_MLP_ROWS = 4,  /* Gaussians the MLP evaluated per light: n, or -- in a sweep of >= 4
                              lights per view without mlp_out -- those blended at some pixel     */
  SSSGS_NCOUNTERS = 8
};

#define SSSGS_TILE 16            /* tiles are 16x16 pixels; part of the tile-list contract   */
#define SSSGS_GBUF_CHANNELS 16   /* see sssgs_out.gbuffer                                    */
#define SSSGS_MAX_TRUNK 8
#define SSSGS_MAX_INC_HIDDEN 2

typedef struct sssgs_ctx sssgs_ctx; /* opaque; owns only scratch memory */

typedef struct {
  int device;             /* CUDA device ordinal                                              */
  int64_t max_gaussians;  /* largest n of any later call                                      */
  int max_width, max_height;
  int64_t max_instances;  /* capacity of the tile-instance list (sum of tiles touched); if it
                             is exceeded the overflow counter is set, nothing is written out
                             of bounds, and the frame is undefined (no host sync happens)     */
  int max_lights_per_pass;/* lights composited per list walk: 1, 4 or 8 (0 -> 8)              */
  void* workspace;        /* optional caller-allocated device scratch (>= sssgs_workspace_bytes,
                             256-byte aligned); NULL -> the context allocates its own         */
  size_t workspace_bytes;
  uint32_t flags;         /* reserved, must be 0                                              */
} sssgs_config;

/* Scene: 3D Gaussians {mu, q, s, o} (L59-72) + PBR attributes {b, r, m, n} (L76) +
 * subsurfaceness (L102) + visibility SH (L110-112) + optional extra MLP feature (S2).       */
typedef struct {
  int64_t n;
  const float* means;      /* [n,3] world space                                               */
  const float* scales;     /* [n,3] ACTIVATED (exp already applied)                    (L72)  */
  const float* rotations;  /* [n,4] unit quaternion (w,x,y,z), caller-normalised       (L72)  */
  const float* opacities;  /* [n]   ACTIVATED, in [0,1]                                (L64)  */
  const float* normals;    /* [n,3] unit                                               (L76)  */
  const float* base_color; /* [n,3]                                                    (L76)  */
  const float* roughness;  /* [n]                                                      (L76)  */
  const float* metallic;   /* [n]                                                      (L76)  */
  const float* subsurface; /* [n]   sss in [0,1]                                       (L102) */
  const float* vis_sh;     /* [n,(deg+1)^2] visibility SH coefficients, real basis
                              Y00 = .2820948, Y1{-1,0,1} = .4886025 {y,z,x}            (L112) */
  int vis_sh_degree;       /* 0 or 1                                                          */
  const float* feat;       /* [n,feat_dim] extra per-Gaussian MLP input, may be NULL if 0     */
  int feat_dim;            /* 0..88, multiple of 4 (row = 16-byte aligned)                    */
} sssgs_gaussians;

/* The global MLP Theta (L98-100, L347).  Input row (in_dim = 40 + feat_dim):
 *   [ n(3) | rot(2) = (q_w,q_x), sign-canonical q_w>=0 | scale(3) | w_in(3) | w_out(3) | d(1) |
 *     v(1) | gamma(mu)(24) = for k=0..3 [sin(2^k pi mu_xyz), cos(2^k pi mu_xyz)] | feat(F) ]
 * params: packed fp32 (or bf16), per layer W[out][in] row-major then b[out]; order = trunk
 * layers, SSS head (3 outputs, sigmoid), incident-head hidden layers, incident output (1,
 * ReLU).  Hidden layers use `activation`.  Compute is 16 bit x 16 bit -> fp32 on the tensor cores:
 * weights and every layer input are rounded (RNE) to `compute` = binary16 (default; finite overflow
 * saturates to +-65504) or bf16; accumulation, biases and activations are fp32.  binary16 is the
 * default because the incident-light output is an unbounded ReLU: with bf16 layer inputs it misses the
 * 1e-2 bound of the specification on up to ~1 % of the rows, with binary16 (same tensor-core rate) it
 * stays within 3e-3.  bf16-stored weights convert to binary16 exactly unless
 * they are below 2^-14 in magnitude.
 * All widths must be multiples of 16 and <= 128.
 * precomputed_out: if non-NULL the MLP is skipped and these values are used instead
 * ([n_cam][n_light][n][4], = (L_SSS rgb, L_in)); lets a caller edit the residual (L169) and
 * lets tests feed the rasteriser reference values.                                           */
typedef struct {
  int in_dim;
  int n_trunk;
  int trunk_width[SSSGS_MAX_TRUNK];
  int n_inc_hidden;
  int inc_hidden_width[SSSGS_MAX_INC_HIDDEN];
  int activation;    /* SSSGS_ACT_RELU | SSSGS_ACT_LEAKY_RELU */
  float leaky_slope; /* paper is silent; 0.01 is customary (S14) */
  int dtype;         /* SSSGS_F32 | SSSGS_BF16: storage type of params */
  const void* params;
  size_t params_bytes;
  const float* precomputed_out;
  int compute;       /* SSSGS_COMPUTE_FP16 (0, default) | SSSGS_COMPUTE_BF16 */
} sssgs_mlp;

/* Pinhole camera.  World -> camera: p_c = R p + t (R row-major); the camera looks down +z,
 * x right, y down; pixel k is centred at integer coordinate k.  Everything is precomputed by
 * the caller so that no transcendental is evaluated upstream of a sort key.                  */
typedef struct {
  float R[9], t[3];
  float fx, fy, cx, cy, tan_half_fovx, tan_half_fovy;
  int width, height;
  float znear;
  float bg[3];
} sssgs_camera;

/* Point light at a known position (L110); RGB intensity multiplier (S16). */
typedef struct {
  float position[3];
  float intensity[3];
} sssgs_light;

/* Outputs; NULL = not wanted.  F = n_cam * n_light frames, frame f = cam * n_light + light.
 * gbuffer pixel (16 fp32, UN-normalised accumulations of Eq. 3):
 *   [0] depth [1-3] normal [4-6] base colour [7] roughness [8] metallic [9] sss
 *   [10-12] L_SSS [13] L_in [14] A = sum of weights [15] final transmittance T.               */
typedef struct {
  float* rgb;            /* [F][H][W][3] linear radiance, no tone mapping (S17)               */
  float* gbuffer;        /* [F][H][W][16]                                                     */
  float* aov_diffuse;    /* [F][H][W][3] diffuse illumination before base colour      (L320) */
  float* aov_specular;   /* [F][H][W][3] specular illumination                         (L320) */
  float* mlp_out;        /* [F][n][4] (L_SSS rgb, L_in) per Gaussian                          */
  uint64_t* sorted_keys; /* [n_cam][max_instances] tile<<32 | bits(depth), sorted             */
  uint32_t* sorted_vals; /* [n_cam][max_instances] Gaussian index of each list entry          */
  uint32_t* tile_ranges; /* [n_cam][tiles_y*tiles_x][2] = [begin,end) of each tile's entries  */
  int64_t* counters;     /* [n_cam][SSSGS_NCOUNTERS]                                          */
} sssgs_out;

/* Scratch bytes a context with this configuration needs (0 on invalid configuration). */
size_t sssgs_workspace_bytes(const sssgs_config* cfg);

/* Create / destroy a context.  destroy is NULL-safe and never frees caller memory. */
int sssgs_create(const sssgs_config* cfg, sssgs_ctx** out);
void sssgs_destroy(sssgs_ctx* ctx);

/* Render F = n_cam x n_light frames.  Geometry (projection, sort, tile lists) runs once per
 * camera; the MLP and the light-dependent channels once per (camera, light); up to
 * max_lights_per_pass lights share one walk of the tile lists (OLAT sweeps).
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).                                */
int sssgs_render(sssgs_ctx* ctx, const sssgs_gaussians* g, const sssgs_mlp* mlp,
                 const sssgs_camera* cams, int n_cam, const sssgs_light* lights, int n_light,
                 const sssgs_out* out, uint32_t flags, void* cuda_stream);

/* Same call with HOST buffers: copies the scene and parameters to the device, renders, copies
 * every requested output back and synchronises.  Returns SSSGS_EOVERFLOW if the instance list
 * overflowed.  (The end-to-end entry point: one host->device crossing per call.)             */
int sssgs_render_host(sssgs_ctx* ctx, const sssgs_gaussians* g, const sssgs_mlp* mlp,
                      const sssgs_camera* cams, int n_cam, const sssgs_light* lights, int n_light,
                      const sssgs_out* out, uint32_t flags);

/* Ray-traced per-Gaussian visibility and its SH fit ("we trace
 * rays using a BVH to quickly estimate the visibility for each Gaussian and learn this as a per
 * Gaussian SH visibility term v"; L81).  Produces the `vis_sh` input of sssgs_gaussians.  For every
 * Gaussian i and direction w_k the ray x(t) = mu_i + (t_min + t) w_k, t >= 0, is traced through a
 * BVH over the alpha >= 1/255 supports of all Gaussians; every other Gaussian j acts at the point of
 * its largest response along the ray, with the opacity rule of the rasteriser (Eq. 3):
 *   m2 = min_{t>=0} (x(t)-mu_j)^T Sigma_j^-1 (x(t)-mu_j),  a = min(0.99, o_j exp(-m2/2)) iff >= 1/255,
 *   V_i(w_k) = prod_{j != i} (1 - a), set to 0 below 1e-4;
 *   vis_sh_out[i][lm] = sum_k weights[k] V_i(w_k) Y_lm(w_k)   (basis and order of vis_sh above).
 * With positions != 0 the K entries of `dirs` are points p_k (the known OLAT light positions of L110):
 * the ray of Gaussian i runs towards p_k and ends there, w = (p_k - mu_i) / d, t in [0, d - t_min]
 * (nothing occludes if d <= t_min), and the SH sum uses that per-Gaussian direction.
 * Only means, scales, rotations and opacities of `g` are read (device pointers, n <=
 * max_gaussians).  The call enqueues on `stream`, never synchronises and uses the context's
 * workspace: it must not overlap a render on the same context (same stream, or ordered by the
 * caller).  The tree and the traversal order are deterministic: results are bit-reproducible.
 * Errors: SSSGS_EINVAL (NULL / n_dirs < 1 or > 4096 / sh_degree not 0 or 1 / t_min < 0 or not
 * finite), SSSGS_ECAPACITY (n > max_gaussians), SSSGS_ECUDA.                                   */
typedef struct {
  int n_dirs;            /* K                                                                 */
  const float* dirs;     /* [K,3] unit vectors, or points if positions != 0 (device)          */
  const float* weights;  /* [K] quadrature weights, e.g. 4 pi / K (device)                    */
  float t_min;           /* ray start offset from the Gaussian's centre, world units          */
  int sh_degree;         /* 0 or 1                                                            */
  float* vis_sh_out;     /* [n,(deg+1)^2] (device), required                                  */
  float* vis_out;        /* [n,K] raw visibilities (device), may be NULL                      */
  int positions;         /* 0: dirs are unit directions; 1: dirs are points, rays end there   */
} sssgs_bake;
int sssgs_bake_visibility(sssgs_ctx* ctx, const sssgs_gaussians* g, const sssgs_bake* bake, void* stream);

/* Backward pass of the render path: steps a8 (deferred shading), a7 (compositing), a2 (the MLP) and, with the
 * optional outputs below, a3 (the projection) and a1 (the MLP's input assembly)
 * ("optimize all parameters jointly via raytraced differentiable
 * rendering", L112, L343-349: the training losses are functions of the rendered image and of the
 * rasterised property images).  For ONE camera and its n_light lights, with
 *   L = sum_l < grad_rgb[l], rgb_l >  ( + sum_l < grad_gbuffer_in[l], gbuffer_l >  when grad_gbuffer_in is given )
 * it computes dL/d of: the G-buffer of every light; the MLP outputs per (light, Gaussian); the MLP
 * parameters Theta; and per Gaussian the opacity, the 2-D mean, the conic (inverse 2-D covariance,
 * entries a, b, c of  power = -(a dx^2 + c dy^2) / 2 - b dx dy), the depth, the normal, the base
 * colour, roughness, metalness and subsurfaceness; and, when grad_means / grad_scales / grad_rotations are
 * given, the 2-D mean / conic / depth gradients pushed through the EWA projection (step a3) to the mean,
 * the scale and the rotation.  The forward decisions
 * (alpha >= 1/255, the T' < 1e-4 stop, the 0.99 clamp, ReLUs) are constants of the differentiation.
 * All pointers are DEVICE pointers, 16-byte aligned, fp32; every gradient array is overwritten.
 * gbuffer must be the G-buffer sssgs_render wrote for the same scene, camera and lights.
 * mlp.dtype must be SSSGS_F32 (mlp.precomputed_out, if given, is used for the forward values and
 * grad_params is then left zero).  Shading and compositing backward are fp32.  The MLP backward runs on the
 * tensor cores (binary16 operands, fp32 accumulation: the forward pass of the listed rows is re-evaluated with
 * the forward kernel's arithmetic; dL/d(mlp_out) is scaled by a power of two so that the deltas fit binary16)
 * when mlp.compute is SSSGS_COMPUTE_FP16 and the MLP has no incident-head hidden layers and at most 4 trunk layers;
 * otherwise (bf16 forward operands included: the binary16 re-evaluation would not reproduce that forward pass), or
 * with SSSGS_BACKWARD_FP32, in fp32 on the CUDA cores (forward re-evaluated in fp32).  Per-Gaussian sums use float atomics: results are
 * reproducible to rounding, not bit for bit.  Enqueues on the stream, never synchronises.
 * With n_light = 0 the per-Gaussian and parameter gradients are zeroed and the per-light pointers are not read;
 * with n = 0 grad_gbuffer is zeroed too (grad_gbuffer_in is not added: nothing is composited).  Errors: SSSGS_EINVAL (NULL / misaligned / dtype), SSSGS_ECAPACITY (n, image size). */
typedef struct {
  const float* grad_rgb;     /* [n_light][H][W][3]  dL / d rgb                         (in)          */
  const float* gbuffer;      /* [n_light][H][W][16] the forward call's G-buffer        (in)          */
  float* grad_gbuffer;       /* [n_light][H][W][16] dL / d gbuffer                     (out, required) */
  float* grad_mlp_out;       /* [n_light][n][4]     dL / d (L_SSS rgb, L_in)           (out, required) */
  float* grad_params;        /* [params_bytes / 4]  dL / d Theta, packing of sssgs_mlp.params (out, may be NULL) */
  float* grad_opacity;       /* [n]                                                    (out, required) */
  float* grad_mean2d;        /* [n][2]  dL / d (pix_x, pix_y)                          (out, required) */
  float* grad_conic;         /* [n][3]  dL / d (a, b, c)                               (out, required) */
  float* grad_depth;         /* [n]                                                    (out, required) */
  float* grad_attr;          /* [n][9]  normal (3), base colour (3), roughness, metalness, sss (out, required) */
  /* step a3 differentiated (Eq. 2): the three above pushed through the EWA projection.  All
     three or none (NULL).  The dependence of the MLP INPUTS on them (step a1) is only included when grad_feat /
     grad_vis_sh below are given.                                                                                  */
  float* grad_means;         /* [n][3]  dL / d mu                                      (out, may be NULL)  */
  float* grad_scales;        /* [n][3]  dL / d s (activated scales, as given)          (out, may be NULL)  */
  float* grad_rotations;     /* [n][4]  dL / d q (r, x, y, z), the quaternion as given (out, may be NULL)  */
  /* step a1 differentiated (Eq. 6: the MLP's input row): both or none (NULL); they need the
     three above and the MLP to run (no precomputed_out).  The gradients that reach the Gaussian through the MLP's
     inputs are then ADDED to grad_means / grad_scales / grad_rotations and to the normal in grad_attr; the
     clamp of the visibility to [0, 1] and the sign of the canonical quaternion are constants.                   */
  float* grad_feat;          /* [n][feat_dim]            dL / d feat                   (out, may be NULL)  */
  float* grad_vis_sh;        /* [n][(vis_sh_degree+1)^2] dL / d vis_sh                 (out, may be NULL)  */
  /* Upstream gradient on the G-buffer itself: the losses of PAPER.md L343-349 that act on the rasterised property
     images rather than on rgb (normal vs. depth consistency, mask entropy on A = channel 14, smoothness of
     roughness / metalness / sss / base colour, the incident-light term on channel 13).  Layout and channel order of
     sssgs_out.gbuffer (un-normalised accumulations; channel 15 = final transmittance).  It is added to what reaches
     the G-buffer through rgb -- grad_gbuffer then holds the sum -- and is propagated through the compositing to
     every per-Gaussian gradient, also where grad_rgb is zero.  Must not alias grad_gbuffer.                       */
  const float* grad_gbuffer_in; /* [n_light][H][W][16]                                 (in, may be NULL)   */
  /* The backward pass rebuilds the camera's tile lists with the context's max_instances.  If the instance count
     exceeds it, the lists are truncated and EVERY gradient is undefined: counters (layout of sssgs_out.counters, one
     camera; SSSGS_CNT_MLP_ROWS is 0) reports SSSGS_CNT_OVERFLOW / SSSGS_CNT_SORT_ERROR exactly as the forward call
     does.  Check it after synchronising whenever the forward call's counters were not checked for the same scene,
     camera and list mode (SSSGS_TIGHT_LISTS).                                                                    */
  int64_t* counters;          /* [SSSGS_NCOUNTERS]                                     (out, may be NULL)  */
} sssgs_grads;
int sssgs_render_backward(sssgs_ctx* ctx, const sssgs_gaussians* g, const sssgs_mlp* mlp,
                          const sssgs_camera* cam, const sssgs_light* lights, int n_light,
                          const sssgs_grads* grads, uint32_t flags, void* cuda_stream);

/* The per-Gaussian MLP alone (steps 1 of the path: input assembly + f_Theta, Eq. 6),
 * for callers that must not allocate device memory and therefore cannot use a context.
 *
 * Who that is: code running inside a host program that claimed the whole GPU for its own memory pool at start-up
 * (an inference server, a renderer plug-in host) -- a cudaMalloc issued from a library there fails or steals from
 * the pool's head-room; and code on a latency-critical thread, because cudaMalloc / cudaFree take the driver's
 * allocator lock and may wait for the device to go idle.  sssgs_create does allocate (its workspace unless one is
 * supplied, and always a stream and events), so such callers get this one call that needs no context at all.
 *
 * What it computes: for every Gaussian i < g->n and light l < n_light
 *     mlp_out[(i * n_light + l) * 4 + 0..3] = (L_SSS r, g, b, L_in)
 * with exactly the kernel, operand precision (sssgs_mlp.compute) and per-row arithmetic of sssgs_render: the
 * values are bit-identical to sssgs_out.mlp_out of a render with the same scene, camera and lights.  NOTE the
 * layout: Gaussian-major [n][n_light][4] (the kernel's native one), not sssgs_out.mlp_out's [n_light][n][4]; with
 * n_light = 1 the two coincide, so one call per light yields arrays usable as sssgs_mlp.precomputed_out.
 * Of `g` only means, scales, rotations, normals, vis_sh (+ degree) and feat (+ feat_dim) are read; of `cam` only R
 * and t (the camera position); all pointers inside g / mlp and mlp_out are DEVICE pointers of `device`, 16-byte
 * aligned; cam and lights are HOST structs, read before the call returns.  mlp.precomputed_out must be NULL.
 *
 * The only intermediate the MLP needs in global memory -- the parameters repacked as 16-bit tensor-core operand
 * tiles -- is kept in a fixed array of SSSGS_STATIC_SCRATCH_BYTES that is part of the library image: every GPU on
 * which the library is used holds those bytes from module load until the process ends, whether or not this
 * function is ever called.  The call itself issues no cudaMalloc / cudaFree and calls no allocating library
 * routine; it enqueues two kernels on `cuda_stream` and returns without synchronising.
 *
 * Limits (beyond them: SSSGS_ECAPACITY and a message naming the limit, nothing is enqueued):
 *   - the packed operands of the network (see build rule in DESIGN.md "MLP stages"; 148 KB for four 128-wide
 *     trunk layers on a 64-wide input) must fit SSSGS_STATIC_SCRATCH_BYTES = 192 KB.  sssgs_render accepts
 *     networks up to ~225 KB; those between need a context;
 *   - n_light <= SSSGS_STATIC_MAX_LIGHTS = 8 per call (one light batch); g->n <= 2^30.
 *
 * First call on a device: looks up the array's device address and the SM count of `device` (a driver query, no
 * allocation) and caches them for the life of the process.  Make that first call at start-up, outside any stream
 * capture; later calls skip the lookup.
 *
 * Sharing: there is ONE array per GPU, used by every call from every thread, and it keeps whatever the last call
 * packed into it.  Each call rewrites all the bytes its own network's tiles occupy before its MLP kernel reads
 * them, so nothing needs clearing between calls and a smaller network after a larger one is fine.  But two calls
 * whose kernels can run at the same time on one GPU (different streams without an ordering between them, or two
 * host threads) race on the array and produce garbage: order them on one stream or with events.  A context-based
 * sssgs_render does not touch the array and may overlap freely.
 *
 * Errors (text via sssgs_last_error(NULL)): SSSGS_EINVAL (NULL / misaligned pointer, architecture rules of
 * sssgs_mlp, device ordinal outside [0, 64)), SSSGS_ECAPACITY (limits above), SSSGS_EARCH (not an sm_100 device),
 * SSSGS_ECUDA.  With g->n = 0 or n_light = 0 the call validates its arguments and does nothing.                  */
#define SSSGS_STATIC_SCRATCH_BYTES (192 * 1024)
#define SSSGS_STATIC_MAX_LIGHTS 8
int sssgs_mlp_eval_static(int device, const sssgs_gaussians* g, const sssgs_mlp* mlp, const sssgs_camera* cam,
                          const sssgs_light* lights, int n_light, float* mlp_out, void* cuda_stream);

/* Relighting from a precomputed reflectance field ("To speed up generation we can
 * precompute a reflectance field assuming white light.  We compute the relit view as the sum over the reflectance
 * field scaled by the environment illumination."):
 *     out[p][c] = sum_{l < n_light} weights[l][c] * frames[l][p][c],      p < n_pixels, c = r, g, b
 * frames  [n_light][n_pixels][3]: the OLAT frames of one view (sssgs_out.rgb of a render with white unit-intensity
 *         lights; render them on a black background -- every frame carries its own (1 - A) bg term and the sum does
 *         not remove it), DEVICE, 16-byte aligned;
 * weights [n_light][3]: RGB radiance the environment sends from light l's direction, DEVICE;
 * out     [n_pixels][3], DEVICE, 16-byte aligned, must not overlap frames.
 * fp32, lights accumulated in order with fused multiply-adds.  One streaming kernel (12 (n_light + 1) n_pixels
 * bytes of HBM traffic), no context, no scratch, no allocation; enqueues on the stream, never synchronises.  With
 * n_light = 0 out is zeroed.  Errors (text via sssgs_last_error(NULL)): SSSGS_EINVAL, SSSGS_ECAPACITY (n_pixels >
 * 2^40 / 12), SSSGS_EARCH, SSSGS_ECUDA.                                                                          */
int sssgs_relight(int device, const float* frames, int n_light, int64_t n_pixels, const float* weights, float* out,
                  void* cuda_stream);

/* Per-stage device timing (measurement aid, off by default).  When enabled, sssgs_render
 * records CUDA events around each stage on the caller's stream (not capture-safe while on);
 * sssgs_profile_read synchronises those events and writes the milliseconds each stage of the
 * LAST call took, summed over cameras and light batches, and the number of kernels per stage. */
enum {
  SSSGS_STAGE_PACK = 0,       /* attribute + weight packing                    */
  SSSGS_STAGE_PROJECT = 1,    /* a3                                            */
  SSSGS_STAGE_DEPTH_SORT = 2, /* a5, Gaussians by depth                        */
  SSSGS_STAGE_EMIT = 3,       /* a4                                            */
  SSSGS_STAGE_TILE_SORT = 4,  /* a5, instances by tile                         */
  SSSGS_STAGE_RANGES = 5,     /* a6 (+ optional list export)                   */
  SSSGS_STAGE_MLP = 6,        /* a1 + a2                                       */
  SSSGS_STAGE_RASTER = 7,     /* a7 + a8: the per-light-batch walks            */
  SSSGS_STAGE_PREPASS = 8,    /* light sweeps: visibility pre-pass of a view (fills the weight cache) + compaction */
  SSSGS_NSTAGES = 9
};
int sssgs_profile_enable(sssgs_ctx* ctx, int enable);
int sssgs_profile_read(sssgs_ctx* ctx, float* stage_ms /* [SSSGS_NSTAGES] */,
                       int* stage_launches /* [SSSGS_NSTAGES], may be NULL */);

/* Number of kernels the last sssgs_render / sssgs_render_host call launched. */
int64_t sssgs_last_launch_count(const sssgs_ctx* ctx);

/* Description of the last error on this context (or of the last failed create if ctx = NULL). */
const char* sssgs_last_error(const sssgs_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* SSSGS_H_ */
