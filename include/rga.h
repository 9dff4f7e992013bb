/* rga.h -- C ABI of the B200 (sm_100a) per-frame forward render of arXiv 2407.10707
 * ("Interactive Rendering of Relightable and Animatable Gaussian Avatars").
 *
 * Problem statement: an avatar A = {M, G, L} -- canonical mesh M with per-vertex attributes, Gaussians G
 * near the mesh, light probes L -- is rendered to an image I' for a novel pose, a new environment map and a viewpoint.
 * Test-time flow (Fig.1 :84): skin -> visibility -> shade -> splat.  One call per stage:
 *
 *   avatar_load        L0  KNN sets S_g (K_g=3), S_v (K_v=19) and Eq.1 interpolation of the pose-independent
 *                          attributes
 *   pose_skin          H1/H2 forward LBS of mesh and Gaussians
 *   visibility_raster  H3/H4 orthographic mesh rasterisation per light direction, then either the shadow-map depth
 *                          test (mode 0, BASELINE.json north_star (b)) or the paper's triangle-ID
 *                          visibility with the median/median/mean filters (mode 1, Eq.3-4)
 *   shade_gaussians    H5  Eq.2 with the Appendix-A BRDF, then gamma
 *   splat_render       H6-H10 back-face opacity kill and the 3DGS tile rasteriser
 *   rga_render_frame   the four per-frame calls as one, independent stages overlapped on a second stream
 *
 * Beyond the per-frame path (each documented at its declaration): splat_attribute (albedo / normal maps), displacement_mlp
 * (d(x, theta) on the tensor cores), gaussians_update (per-frame KNN + Eq.1 for moved Gaussians), densify_density
 * (Algorithm 1), and the training side of one view: image_loss (Eq.5), regularisers (Eq.6-9), splat_backward,
 * shade_backward, pose_backward (the backward of H10 + H6, of H5, and of H2 + Eq.1).
 *
 * Conventions
 *  - Every pointer marked "dev" is DEVICE memory owned by the caller (row-major, fp32 / int32); pointers marked "host"
 *    are host memory read during the call.  The library never frees or keeps caller pointers after avatar_load returns
 *    (it copies what it needs), except that per-frame calls read their dev arguments asynchronously on `stream`, so
 *    the caller keeps them alive until the stream has passed the call.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  The four per-frame calls only enqueue
 *    work: no allocation, no host synchronisation, no host-side data-dependent size, so a frame can be captured into
 *    a CUDA graph.  All scratch is allocated in avatar_load at the declared maxima.
 *  - Errors: every call returns an rga_status; nothing throws across the ABI.  rga_last_error() gives a thread-local
 *    message.  Device-side capacity overflow (more (Gaussian,tile) duplicates than max_duplicates) sets a sticky
 *    device status word that rga_check() reads back; the frame's image is then undefined.
 *  - Calling a stage before its producer in the same pose returns RGA_ERR_STATE.
 *  - Concurrency: an rga_avatar owns its scratch and its stage state, so calls on ONE handle must be ordered (one host thread
 *    at a time, work enqueued on one stream at a time, or streams ordered by events).  Different handles share nothing and may
 *    be used from different threads and streams at once (tests/test_gpu_parity.py renders two at once, bit-identical to serial).
 *  - Quaternions are (w,x,y,z).  World is z-up.  Camera looks down +z, x right, y down; image origin top-left;
 *    pixel (i,j) samples at (i+1/2, j+1/2).  Bone matrices are posed-global x inverse-bind, row-major 3x4.
 *  - There is no CPU fallback: without a CUDA device every entry point that computes returns RGA_ERR_CUDA.
 */
#ifndef RGA_H_
#define RGA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define RGA_API __attribute__((visibility("default")))
#else
#define RGA_API
#endif

typedef struct rga_avatar rga_avatar; /* opaque; owns all device scratch */

typedef enum {
  RGA_OK = 0,
  RGA_ERR_INVALID_ARG = 1,
  RGA_ERR_CUDA = 2,
  RGA_ERR_OOM = 3,
  RGA_ERR_STATE = 4,
  RGA_ERR_CAPACITY = 5
} rga_status;

/* avatar_load input.  PAPER.md:86 lists the vertex attributes {r,s,a,gamma,p,w,n,dx}; PAPER.md:88 the Gaussians. */
typedef struct {
  int32_t n_verts, n_faces, n_bones, n_gauss;   /* n_verts < 2^21, n_faces < 2^24 (packed faces).  Beyond about 45k vertices the
                                                    rasteriser's table of snapped coordinates moves from shared memory to an
                                                    L2-resident scratch buffer (slower, same results)                    */
  int32_t k_g;                 /* neighbours per Gaussian, 1..3 (paper: 3)          */
  int32_t k_v;                 /* neighbours per vertex, odd, 1..31 (paper: 19); clamped to n_verts */
  const float*   vert_pos;     /* dev [n_verts][3]  canonical x                                      */
  const int32_t* faces;        /* dev [n_faces][3]                                                   */
  const float*   vert_normal;  /* dev [n_verts][3]  unit normals n, or NULL = area-weighted normals of the canonical mesh,
                                  computed once here (sum of (x_b-x_a) x (x_c-x_a) over a vertex's faces in ascending face
                                  order, normalised; a vertex without a face gets 0; readable as RGA_BUF_VERT_NORMAL;
                                  DESIGN.md reading A40)                                              */
  const float*   vert_skin_w;  /* dev [n_verts][n_bones] LBS weights w, rows sum to 1                */
  const float*   vert_disp;    /* dev [n_verts][3]  static average displacement or NULL = 0 */
  const float*   vert_albedo;  /* dev [n_verts][3]  a                                                */
  const float*   vert_rough;   /* dev [n_verts]     gamma in (0, 1].  The radiance tolerance (2e-3 of max(1, L_o)) is met for
                                  gamma >= 0.07; mirror-like values lose it to fp32 (gamma = 0.01: up to 4e-3 under a
                                  strongly HDR map -- the half vector's tangential part is a difference of unit vectors) */
  const float*   vert_spec;    /* dev [n_verts]     specular tint p                                  */
  const float*   gauss_pos;    /* dev [n_gauss][3]  canonical x_g                                    */
  const float*   gauss_quat;   /* dev [n_gauss][4]  (w,x,y,z), any non-zero norm; NULL = interpolate vert_quat  */
  const float*   gauss_scale;  /* dev [n_gauss][3]; NULL = interpolate vert_scale                        */
  const float*   gauss_opacity;/* dev [n_gauss] or NULL = 1 ("always set the opacity ... to 1") */
  int32_t max_width, max_height;   /* largest camera this avatar will be rendered with                 */
  int32_t max_vis_dirs;            /* largest K_vis (multiple of 32 not required)                      */
  int32_t max_vis_res;             /* largest depth-map side R_v, <= 256 (snapped raster coordinates are 16-bit) */
  int32_t max_env_texels;          /* largest rows*cols of an environment map                           */
  int64_t max_duplicates;          /* capacity of the (tile,depth) key buffers; 0 = library picks       */
  /* The paper's own layout: rotation r and scale s are VERTEX attributes interpolated to the Gaussians
   * by Eq.1 like every other attribute.  Used when gauss_quat / gauss_scale is NULL (reading A2): neighbour
   * quaternions are first given the sign of the nearest neighbour's (q and -q are the same rotation), then averaged with the
   * Eq.1 weights; the result is normalised where it is used (H2). */
  const float*   vert_quat;    /* dev [n_verts][4] (w,x,y,z) or NULL                                  */
  const float*   vert_scale;   /* dev [n_verts][3] or NULL                                            */
} rga_avatar_desc;

typedef struct {
  float R_wc[9];   /* row-major world->camera rotation */
  float t_wc[3];
  float fx, fy, cx, cy;
  int32_t width, height;
  float z_near;    /* Gaussians with camera z <= z_near are culled (3DGS: 0.2) */
} rga_camera;

typedef struct {
  int32_t n_dirs;            /* K_vis                                                                   */
  int32_t res;               /* R_v: depth maps are res x res                                           */
  int32_t mode;              /* 0 = shadow-map depth test, 1 = paper (triangle-ID + Eq.3-4 filters)     */
  const float* dirs;         /* dev [n_dirs][3] unit vectors pointing TOWARD the light                  */
  float depth_bias_texels;   /* mode 0: slope-scaled bias, in depth-map texels (default 1)              */
  float depth_bias_world;    /* mode 0: constant bias in world units (default 0.015)                    */
  float slope_max;           /* mode 0: clamp of the slope factor tan(theta) (default 8)                */
  int32_t keep_maps;         /* non-zero: also keep the triangle-ID maps in mode 0 (parity / debug)     */
  int32_t cull_backfaces;    /* non-zero: the mesh is CLOSED with outward counter-clockwise faces, so the surface
                                nearest a light is always a face turned towards it: triangles whose snapped light-space
                                area is negative are skipped (reading A36).  On such a mesh the maps differ from
                                the unculled ones only where a nearly edge-on back face extrapolates its plane in front of
                                the surface (< 1 % of the covered texels).  0 = rasterise every triangle                */
} rga_vis_params;

typedef struct {
  int32_t rows, cols;              /* equirectangular, z-up; texel (i,j) centre theta=(i+1/2)pi/rows, phi=(j+1/2)2pi/cols */
  const float* radiance;           /* dev [rows][cols][3]                                                */
  const int32_t* texel_to_dir;     /* dev [rows*cols] visibility direction used by each texel, or NULL = identity */
  float gamma;                     /* colour = clamp(L_o,0,1)^(1/gamma)                                   */
  int32_t use_visibility;          /* 0 = ignore visibility (v = 1; the paper's "no visibility" variant) */
} rga_env;

/* L0.  Copies / derives everything it needs from `desc`; allocates all scratch.  Synchronises `stream` before it
 * returns.  *out is NULL on failure. */
RGA_API rga_status avatar_load(const rga_avatar_desc* desc, void* stream, rga_avatar** out);
RGA_API rga_status avatar_free(rga_avatar* av);

/* H1 + H2.  bone_mats: dev [n_bones][12].  Produces posed vertices/normals, posed Gaussians/normals/covariances and
 * the orthographic window (centre, radius) used by every light direction. */
RGA_API rga_status pose_skin(rga_avatar* av, const float* bone_mats, void* stream);

/* H3 + H4.  Needs pose_skin.  Produces per-Gaussian visibility bits (mode 0) or per-vertex counts 0..k_v (mode 1). */
RGA_API rga_status visibility_raster(rga_avatar* av, const rga_vis_params* params, void* stream);

/* H5.  Needs pose_skin, and visibility_raster unless env->use_visibility == 0.  cam_pos: host float[3]. */
RGA_API rga_status shade_gaussians(rga_avatar* av, const rga_env* env, const float cam_pos[3], void* stream);

/* H6-H10.  Needs shade_gaussians.  bg: host float[3].  out_image: dev [height][width][3] fp32, caller-owned. */
RGA_API rga_status splat_render(rga_avatar* av, const rga_camera* cam, const float bg[3], float* out_image, void* stream);

/* Moving Gaussians (the paper's training / editing regime, where x_g are free parameters and the KNN step is repeated
 * every frame -- PAPER.md:88-93, Table 4 "KNN" :300-302): recomputes S_g (K_g nearest canonical vertices of every new
 * position), the Eq.1 weights and every interpolated attribute {n, a, gamma, p, w, dx} exactly as avatar_load does; rotation,
 * scale and opacity are kept.  gauss_pos: dev [n_gauss][3].  Enqueue-only; call pose_skin afterwards. */
RGA_API rga_status gaussians_update(rga_avatar* av, const float* gauss_pos, void* stream);

/* Backward of splat_render (training / editing regime, PAPER.md:128 "the same image loss as 3DGS", :185): for the frame
 * last rendered by splat_render or rga_render_frame with THIS camera and background, image = the out_image that call
 * wrote (unchanged) and dL_dimage = dL/d(out_image) (both dev [height][width][3] fp32), the gradient of L with respect to every Gaussian's splatted colour c_g, opacity o_g,
 * posed mean xbar_gd and posed 3D covariance (the 6 unique entries xx,xy,xz,yy,yz,zz; an off-diagonal entry's gradient
 * counts both of its positions).  The forward's discrete decisions are frozen: tile lists and their order, culled
 * Gaussians (rows of zeros), per-pixel skips (power > 0, alpha < 1/255) and the stopping entry; where alpha is clamped
 * to 0.99 no gradient reaches opacity, mean or covariance (reading A32).  The dependence of the colour on the
 * position through shading is NOT included (that is the backward of shade_gaussians).
 * Outputs are DEVICE buffers, each may be NULL: out_dcolor [n_gauss][3], out_dopacity [n_gauss], out_dmean [n_gauss][3],
 * out_dcov [n_gauss][6].  dL/dmu2D and dL/dconic stay readable through RGA_BUF_SPLAT_GRAD.  Enqueue-only. */
RGA_API rga_status splat_backward(rga_avatar* av, const rga_camera* cam, const float bg[3], const float* image, const float* dL_dimage,
                                  float* out_dcolor, float* out_dopacity, float* out_dmean, float* out_dcov, void* stream);

/* Backward of shade_gaussians (the material / lighting side of training): for the shading last
 * computed by shade_gaussians or rga_render_frame with THIS env and cam_pos, and dL_dcolor = dL/d(colour) per Gaussian
 * (dev [n_gauss][3], e.g. splat_backward's out_dcolor), the gradient of L with respect to every Gaussian's albedo
 * a_g, roughness gamma_g, specular p_g, posed normal n_gd (as a free 3-vector) and posed position (through w_o only),
 * and with respect to the environment map L.  Visibility is a frozen input.  colour = clamp(L_o, 0, 1)^(1/gamma) has
 * derivative 0 at and beyond the clamp limits (reading A33), so a Gaussian whose radiance is 0 (hidden,
 * facing away) or >= 1 in a channel gets no gradient from that channel.
 * Outputs are DEVICE buffers, each may be NULL: out_dalbedo [n_gauss][3], out_drough [n_gauss], out_dspec [n_gauss],
 * out_dnormal [n_gauss][3], out_dpos [n_gauss][3], out_denv [rows][cols][3].  Environment maps of more than 5,030 texels
 * (46 bytes per texel of shared memory) are refused with RGA_ERR_INVALID_ARG; the forward calls take up to 6,595.
 * Enqueue-only. */
RGA_API rga_status shade_backward(rga_avatar* av, const rga_env* env, const float cam_pos[3], const float* dL_dcolor,
                                  float* out_dalbedo, float* out_drough, float* out_dspec, float* out_dnormal, float* out_dpos,
                                  float* out_denv, void* stream);

/* Eq.5: L_img = (1 - lambda) L_1 + lambda L_D-SSIM between a rendered image and its target, both DEVICE
 * [height][width][3] fp32, width <= max_width and height <= max_height of the avatar (whose scratch it uses), with the
 * gradient dL_img/d(image) -- the dL_dimage of splat_backward.  L_1 = mean |I - I^|; L_D-SSIM = 1 - SSIM with the 11x11
 * Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2, averaged over pixels and channels, as in 3DGS
 * (reading A34); the paper's lambda is 0.2.  out_loss: dev f32 [3] = {L_img, L_1, SSIM} or NULL;
 * out_dL_dimage: dev [height][width][3] or NULL.  Enqueue-only. */
RGA_API rga_status image_loss(rga_avatar* av, const float* image, const float* target, int width, int height, float lambda,
                              float* out_loss, float* out_dL_dimage, void* stream);

/* image_loss without an avatar handle and WITHOUT ANY ALLOCATION (Eq.5; same kernels, same arithmetic, same
 * arguments as image_loss): for callers that cannot call cudaMalloc -- code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it.  Its scratch (nine floats per pixel + two accumulators) is a fixed device array inside the
 * library: width * height <= RGA_IMAGE_LOSS_STATIC_MAX_PIXELS (262,144 = 512 x 512), larger images are refused with
 * RGA_ERR_INVALID_ARG and a message; every GPU that loads the library holds the array's 9.0 MiB until the process exits.
 * The call makes no cudaMalloc / cudaFree and calls no allocating library routine; it enqueues one 16-byte memset and up
 * to three kernels on `stream` (device of the current context).  ALL calls share the one array, which keeps the last call's
 * contents (everything a call reads is rewritten by that call first): calls on the same stream are ordered and safe; calls
 * that overlap on the GPU (different streams, or several host threads on different streams) RACE -- serialise them.
 * image, target: dev [height][width][3]; out_loss: dev f32 [3] = {L_img, L_1, SSIM} or NULL; out_dL_dimage: dev
 * [height][width][3] or NULL.  Enqueue-only. */
#define RGA_IMAGE_LOSS_STATIC_MAX_PIXELS 262144
RGA_API rga_status rga_image_loss_static(const float* image, const float* target, int width, int height, float lambda,
                                         float* out_loss, float* out_dL_dimage, void* stream);

/* Regularisers of the training objective Eq.10, evaluated on the avatar's own tables, each as the plain
 * sum the paper writes (the lambdas of Eq.10 are the caller's), with gradients:
 *   Eq.6 L_smooth = sum_i sum_{k in S_v^i} ||*^i - *^k||_1 over the vertex attributes * in {albedo, roughness, specular};
 *   Eq.7 L_mdist  = sum_i sum_{k in S_g^i} ||x_g^i - x^k||_2  (canonical Gaussian positions vs their K_g vertices);
 *   Eq.8 L_disp   = sum_i ||dx^i||_2  (the current per-vertex displacement: displacement_mlp's if it ran, else the static one);
 *   Eq.9 L_scale  = sum_i max(0, s_g^i - s0) over the three scale components; the paper's s0 is 0.005.
 * Slopes at the kinks (equal attributes, zero distance or displacement, s = s0) are 0 (reading A35).
 * out_losses: dev f32 [4] = {L_smooth, L_mdist, L_disp, L_scale} or NULL.  Gradient outputs, DEVICE, each may be NULL:
 * out_dalbedo [n_verts][3], out_drough [n_verts], out_dspec [n_verts] (Eq.6); out_dgauss_pos [n_gauss][3] (Eq.7);
 * out_ddisp [n_verts][3] (Eq.8); out_dscale [n_gauss][3] (Eq.9).  Enqueue-only. */
RGA_API rga_status regularisers(rga_avatar* av, float s0, float* out_losses, float* out_dalbedo, float* out_drough, float* out_dspec,
                                float* out_dgauss_pos, float* out_ddisp, float* out_dscale, void* stream);

/* Backward of pose_skin's Gaussian half (H2) and of Eq.1: pulls a frame's posed-space gradients back to the canonical
 * parameters the paper optimises.  Inputs (DEVICE, each may be NULL = zero): d_mean [n_gauss][3]
 * and d_mean2 [n_gauss][3], summed = dL/d xbar_gd (splat_backward's out_dmean and shade_backward's out_dpos), d_normal [n_gauss][3] = dL/d nbar_gd
 * (shade_backward's out_dnormal), d_cov [n_gauss][6] (splat_backward's out_dcov), and the per-Gaussian material gradients
 * d_albedo [n_gauss][3], d_rough, d_spec [n_gauss] (shade_backward's).  bone_mats: dev [n_bones][12], the pose of that
 * frame.  Outputs (DEVICE, each may be NULL): d_gauss_pos [n_gauss][3] (canonical x_g), d_gauss_quat [n_gauss][4] (w,x,y,z;
 * the forward normalises q, so the gradient is tangent to it), d_gauss_scale [n_gauss][3], d_bones [n_bones][12] (the pose,
 * :155), and through the transpose of Eq.1 -- S_g and its weights frozen -- the vertex attributes d_vert_disp [n_verts][3]
 * (dx), d_vert_normal [n_verts][3] (n, incl. the renormalisation of the interpolated normal), d_vert_albedo [n_verts][3],
 * d_vert_rough, d_vert_spec [n_verts].  The skinning weights are not differentiated.  k_g <= 8.  Enqueue-only. */
typedef struct { const float *d_mean, *d_mean2, *d_normal, *d_cov, *d_albedo, *d_rough, *d_spec; } rga_posed_grads;
typedef struct {
  float *d_gauss_pos, *d_gauss_quat, *d_gauss_scale, *d_bones, *d_vert_disp, *d_vert_normal, *d_vert_albedo, *d_vert_rough, *d_vert_spec;
} rga_canonical_grads;
RGA_API rga_status pose_backward(rga_avatar* av, const float* bone_mats, const rga_posed_grads* in, const rga_canonical_grads* out,
                                 void* stream);

/* Algorithm 1, "Gaussian densification based on density": from the avatar's current
 * S_g (avatar_load / gaussians_update) and its mesh, counts the Gaussians near every vertex (D_v), estimates the Gaussian
 * density of every triangle d_f = sum of its three D_v / (6 K_g), sets P = max(0, d0 - d_f), asks for
 * N' = floor(sum(P) * p0) new Gaussians, draws their triangles by multinomial sampling from P / sum(P) and places each
 * uniformly at random on its triangle of the CANONICAL mesh.  The paper's values are d0 = 1, p0 = 0.02.
 * The random numbers are the caller's: rnd, dev uint32 [3 * max_out], raw 32-bit draws -- rnd[3j] picks the triangle of
 * new Gaussian j (inverse CDF), rnd[3j+1] and rnd[3j+2] place it (readings A29-A31 fix the arithmetic).
 * out_pos: dev f32 [max_out][3]; out_tri: dev i32 [max_out] or NULL; out_count: dev i32 [1] or NULL, receives N'.
 * min(N', max_out) entries are written, in draw order.  D_v, P, n_g and {sum(P), N'} stay readable through
 * rga_get_buffer (RGA_BUF_DENS_*).  Enqueue-only; the avatar itself is not changed: append the positions to the
 * Gaussian set and load (or gaussians_update) again.  Requires 0 < d0 <= 32768 and p0 >= 0. */
RGA_API rga_status densify_density(rga_avatar* av, float d0, float p0, const uint32_t* rnd, int max_out, float* out_pos,
                                   int32_t* out_tri, int32_t* out_count, void* stream);

/* Displacement network d(x, theta): dx_i = MLP([gamma(x_i), theta]) for every canonical vertex, with
 * gamma(x) = [sin(2 pi B x), cos(2 pi B x)] (random Fourier features, B = rff), four hidden layers of width 256 with ReLU
 * and a linear 256 -> 3 head (readings A26-A28).  Runs on the tensor cores (tcgen05, TF32 operands, fp32
 * accumulation); the result replaces the avatar's displacement attribute: vertices become x + dx, Gaussians x_g + Eq.1(dx),
 * exactly as avatar_load does with a static displacement.  Call pose_skin (or rga_render_frame) afterwards.
 * All pointers are DEVICE memory, row-major fp32; W1's columns are [sin block | cos block | theta]. */
typedef struct {
  int32_t n_freq;             /* F = rows of B; a multiple of 16 in [16, 128]                         */
  int32_t n_pose;             /* length of theta (72 in the paper)                                    */
  const float* rff;           /* dev [F][3]                                                           */
  const float* W1;            /* dev [256][2 F + n_pose]                                              */
  const float* b1;            /* dev [256]                                                            */
  const float* Wh;            /* dev [3][256][256]  layers 2..4                                       */
  const float* bh;            /* dev [3][256]                                                         */
  const float* Wo;            /* dev [3][256]                                                         */
  const float* bo;            /* dev [3]                                                              */
} rga_disp_mlp;
RGA_API rga_status displacement_mlp(rga_avatar* av, const rga_disp_mlp* mlp, const float* theta, void* stream);

/* Back to the static per-vertex displacement given to avatar_load (NULL = 0) after displacement_mlp: x + dx for
 * the mesh and Eq.1 of dx over the current S_g for the Gaussians, bit-identical to a fresh load.  Enqueue-only; call pose_skin
 * afterwards.  (gaussians_update keeps whichever displacement is current: after displacement_mlp it re-interpolates the
 * network's dx over the new neighbour sets.) */
RGA_API rga_status displacement_static(rga_avatar* av, void* stream);

/* Attribute maps: the same splat (H6-H10, incl. the back-face opacity kill) with the Gaussian's albedo a_g
 * (RGA_ATTR_ALBEDO; the albedo map of PAPER.md:177 and :239) or its posed normal n_gd, signed components
 * (RGA_ATTR_NORMAL; the normal maps behind the paper's normal-error metric) as the splatted colour.  Needs
 * pose_skin only; no visibility, no shading.  out_image: dev [height][width][3] fp32; pixels not covered get bg. */
#define RGA_ATTR_ALBEDO 1
#define RGA_ATTR_NORMAL 2
RGA_API rga_status splat_attribute(rga_avatar* av, const rga_camera* cam, const float bg[3], int which, float* out_image,
                                   void* stream);

/* One whole frame: pose_skin, visibility_raster (skipped when vis == NULL, which needs
 * env->use_visibility == 0), shade_gaussians and splat_render with the same arguments, results and intermediates as the
 * four calls above.  Enqueue-only like them.  The steps that depend neither on visibility nor on shading (H6-H9 and
 * the environment table) are issued on a second stream owned by the avatar and joined before the blend, so `stream`
 * observes the whole frame in order; the call can be captured into a CUDA graph.
 * One difference in the intermediates: this call knows the camera when it tests visibility, so in mode 0 the depth test
 * is not run for Gaussians that face away from the camera (their opacity is 0 and shade_gaussians skips
 * them by the same test); their RGA_BUF_VISBITS words are 0.  Where the light-frame and environment tables fit shared memory
 * (n_dirs <= 2,048, rows * cols <= 4,096 and 48 n_dirs + 24 rows * cols + 13 KB within 226 KB) depth test and shading run as one
 * kernel that also leaves out the directions none of whose texels can light the Gaussian (n . w_i <= 0 for all of them); those
 * bits are 0 as well.  Larger tables fall back to the two kernels of the separate calls, which test every direction of a
 * camera-facing Gaussian.  Radiance, colour and image are unchanged.  To shade the
 * same pose from ANOTHER camera afterwards, call visibility_raster first (shade_gaussians returns RGA_ERR_STATE if not). */
RGA_API rga_status rga_render_frame(rga_avatar* av, const float* bone_mats, const rga_vis_params* vis, const rga_env* env,
                                    const float cam_pos[3], const rga_camera* cam, const float bg[3], float* out_image,
                                    void* stream);

/* Intermediates (parity tests, debugging).  Layouts are documented next to each id. */
typedef enum {
  RGA_BUF_KNN_G = 0,          /* i32 [n_gauss][k_g]                                  */
  RGA_BUF_UBAR_G = 1,         /* f32 [n_gauss][k_g]  normalised Eq.1 weights         */
  RGA_BUF_KNN_V = 2,          /* i32 [n_verts][k_v]                                  */
  RGA_BUF_GAUSS_STATIC = 3,   /* f32 [n_gauss][16]: xbar(3) pad, n(3) pad, albedo(3) rough, spec pad pad pad */
  RGA_BUF_GAUSS_SKIN_W = 4,   /* f32 [n_gauss][n_bones]                              */
  RGA_BUF_VERT_POSED = 5,     /* f32 [n_verts][4]  x' (xyz, w unused)                */
  RGA_BUF_VERT_NORMAL_POSED = 6, /* f32 [n_verts][4]                                 */
  RGA_BUF_GAUSS_POSED = 7,    /* f32 [n_gauss][4]  xbar_gd                           */
  RGA_BUF_GAUSS_NORMAL_POSED = 8, /* f32 [n_gauss][4] n_gd                           */
  RGA_BUF_GAUSS_COV = 9,      /* f32 [n_gauss][6]  xx,xy,xz,yy,yz,zz                 */
  RGA_BUF_WINDOW = 10,        /* f32 [4]  centre xyz, radius                         */
  RGA_BUF_ZMAP = 11,          /* u32 [n_dirs][res][res] float bits of depth, 0xFFFFFFFF = empty */
  RGA_BUF_IDMAP = 12,         /* i32 [n_dirs][res][res] winning triangle, -1 = empty (mode 1 or keep_maps) */
  RGA_BUF_VISBITS = 13,       /* u32 [n_gauss][ceil(n_dirs/32)]  bit (k%32) of word k/32 */
  RGA_BUF_VCOUNT = 14,        /* u8  [n_verts][n_dirs]  mean-filter numerators 0..k_v (mode 1) */
  RGA_BUF_RADIANCE = 15,      /* f32 [n_gauss][4]  linear L_o rgb, w unused          */
  RGA_BUF_COLOR = 16,         /* f32 [n_gauss][4]  gamma-corrected colour            */
  RGA_BUF_MU2D = 17,          /* f32 [n_gauss][2]                                    */
  RGA_BUF_DEPTH = 18,         /* f32 [n_gauss]                                       */
  RGA_BUF_CONIC_OPACITY = 19, /* f32 [n_gauss][4]                                    */
  RGA_BUF_RECT = 20,          /* i32 [n_gauss][4]  x0,y0,x1,y1 (tiles, half-open)    */
  RGA_BUF_TOUCHED = 21,       /* u32 [n_gauss]                                       */
  RGA_BUF_NUM_DUPLICATES = 22,/* u32 [1]  D                                          */
  RGA_BUF_KEYS_SORTED = 23,   /* u64 [D]  tile << 32 | depth bits                    */
  RGA_BUF_VALS_SORTED = 24,   /* u32 [D]  Gaussian index                             */
  RGA_BUF_TILE_RANGES = 25,   /* u32 [tiles][2]                                      */
  RGA_BUF_T_FINAL = 26,       /* f32 [height][width]                                 */
  RGA_BUF_N_CONTRIB = 27,     /* u32 [height][width]                                 */
  RGA_BUF_VERT_BITS_RAW = 28, /* u32 [n_verts][ceil(n_dirs/32)] raw vertex visibility (mode 1) */
  RGA_BUF_VERT_DISP = 29,     /* f32 [n_verts][4] per-pose displacement of displacement_mlp (xyz, w unused) */
  RGA_BUF_DENS_DV = 30,       /* i32 [n_verts]  Algorithm 1: Gaussians near each vertex              */
  RGA_BUF_DENS_P = 31,        /* u32 [n_faces]  P = max(0, d0 - d_f) in fixed point (P * 2^16)         */
  RGA_BUF_DENS_NG = 32,       /* i32 [n_faces]  Gaussians added per triangle by the last call          */
  RGA_BUF_DENS_HDR = 33,      /* u64 [2]        sum of the fixed-point P, N'                            */
  RGA_BUF_SPLAT_GRAD = 34,    /* f32 [n_gauss][12] splat_backward: d_colour(3), d_opacity, d_mu2D(2), d_conic(3), pad(3) */
  RGA_BUF_GAUSS_ORDER = 35,   /* i32 [n_gauss] caller index of the i-th Gaussian in the library's internal (spatial) order */
  RGA_BUF_VERT_NORMAL = 36,   /* f32 [n_verts][3] canonical vertex normals as used (the caller's, or the computed ones) */
  RGA_BUF_COUNT_ = 37
} rga_buffer_id;

/* Gaussian order.  PAPER.md:88-93 defines no order of the Gaussians and a trained asset's is arbitrary, so avatar_load sorts
 * them ONCE by the Morton code of their canonical position and keeps the permutation (RGA_BUF_GAUSS_ORDER); gaussians_update
 * keeps it.  Every array the CALLER passes or receives is in the caller's order: the rga_avatar_desc tables, gaussians_update's
 * positions, every [n_gauss] gradient input / output of the backward calls, the Gaussian indices in RGA_BUF_VALS_SORTED
 * (equal (tile, depth) keys order by the caller's index) and whatever rga_read_buffer copies to the host.  Only the DEVICE
 * pointers rga_get_buffer returns for the per-Gaussian buffers ([n_gauss][...] rows above) address the library's internal
 * order: row i belongs to the caller's Gaussian RGA_BUF_GAUSS_ORDER[i].
 *
 * Returns the device pointer and current size in bytes of an internal buffer (valid until the next call that
 * rewrites it).  For data-dependent sizes (KEYS/VALS) this synchronises `stream` to read D. */
RGA_API rga_status rga_get_buffer(rga_avatar* av, int which, void* stream, const void** dev_ptr, size_t* bytes);

/* Copies an internal buffer to HOST memory `host_dst` (capacity bytes), per-Gaussian rows put back into the caller's order;
 * *bytes = size copied.  Synchronises `stream`.
 * RGA_ERR_INVALID_ARG if capacity is too small (then *bytes holds the required size). */
RGA_API rga_status rga_read_buffer(rga_avatar* av, int which, void* stream, void* host_dst, size_t capacity, size_t* bytes);

/* Synchronises `stream` and returns the sticky device status (RGA_OK or RGA_ERR_CAPACITY); clears it. */
RGA_API rga_status rga_check(rga_avatar* av, void* stream);

/* Number of kernels the library has launched since the avatar was loaded (bench.py's gpu_launches claim). */
RGA_API int64_t rga_launch_count(const rga_avatar* av);

/* Optional per-kernel timing.  While enabled, the library records a CUDA event on `stream` after each of its kernels.
 * rga_profile_read synchronises `stream`, writes up to `capacity` entries (names: capacity x 32 chars, ms: elapsed
 * milliseconds of each kernel since the previous event) and clears the log.  Not graph-capturable while enabled.
 * on == 2 (timeline): rga_render_frame keeps its second stream and every entry is the completion time of that kernel since
 * the call began -- how the two streams actually interleave. */
RGA_API rga_status rga_profile_enable(rga_avatar* av, int on);
RGA_API rga_status rga_profile_read(rga_avatar* av, void* stream, char* names, float* ms, int capacity, int* count);

/* Measures the device's FP32 FMA throughput (register-resident FFMA chains on every SM, best of 3, ~5 ms) -- the
 * denominator bench.py quotes beside the ALU-bound kernels.  Synchronises `stream`. */
RGA_API rga_status rga_measure_fp32_peak(void* stream, float* tflops);

RGA_API const char* rga_last_error(void);
RGA_API const char* rga_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RGA_H_ */
