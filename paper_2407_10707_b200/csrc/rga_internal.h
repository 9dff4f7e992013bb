// Internal state and kernel launchers of librga (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/rga.h"

#define RGA_TILE 16
#define RGA_MAX_PROF 96
#define RGA_STATIC_MAX_DEVICES 64   // devices whose static-scratch address rga_image_loss_static remembers
#define RGA_SORT_SMALL 2048      // tiles up to this many entries are sorted in shared memory (bitonic), longer ones by the radix path of the same kernel
#define RGA_SEG 64               // compositing segment: list entries blended by one work item

struct rga_avatar {
  // sizes
  int n_verts, n_faces, n_bones, n_gauss, k_g, k_v;
  int max_w, max_h, max_dirs, max_res, max_env;
  long long max_dup;
  int num_sms;
  // static (load-time) tables
  float4* v_pos;       // [n_verts]  canonical x (displacement_mlp re-derives x + dx from it)
  float4* v_disp;      // [n_verts]  per-pose displacement written by displacement_mlp
  float4* g_pos;       // [n_gauss]  canonical x_g
  // Gaussian order (order_kernels.cu): every per-Gaussian table below is stored in the library's spatial order;
  // g_order[i] = caller index of the i-th Gaussian, g_inv = its inverse; gi_pos = the caller's positions in library order
  int *g_order, *g_inv; float* gi_pos; unsigned* bb_scratch; float* bb_dev;
  // the library's copies of the vertex tables Eq.1 reads (gaussians_update re-interpolates from them)
  float *vt_pos, *vt_disp, *vt_normal, *vt_albedo, *vt_rough, *vt_spec;   // [n_verts][3] x4 (disp NULL = 0), [n_verts] x2
  float *vt_quat, *vt_scale;   // [n_verts][4], [n_verts][3]: the paper's per-vertex rotation / scale when they are interpolated (else NULL)
  float* knn_d2;       // [n_gauss][k_g] squared distances of the last Gaussian KNN
  // uniform grid over the canonical vertices (exact KNN of the Gaussians); grid_G == 0: brute force
  int grid_G; float grid_h, grid_o[3]; unsigned* grid_start; int* grid_verts;
  // Algorithm 1 (density-based densification): D_v, P in fixed point, its running sum, n_g, per-tile sums, {sum, N'}
  int* dens_dv; unsigned* dens_pfix; unsigned long long* dens_cdf; int* dens_ng; unsigned long long* dens_block; unsigned long long* dens_hdr;
  float* mlp_bias1;    // [256] layer-1 bias of the displacement network with the pose folded in
  float4* v_xbar;      // [n_verts]  x + dx
  float4* v_normal;    // [n_verts]
  float* v_skin_w;     // [n_verts][B]
  int* faces;          // [n_faces][3]
  unsigned long long* faces_packed;  // [n_faces] 3 x 21-bit vertex indices (one 8-byte load per triangle)
  int* knn_v;          // [n_verts][k_v]
  int* knn_g;          // [n_gauss][k_g]
  float* ubar_g;       // [n_gauss][k_g]
  float4* g_static;    // [n_gauss][4]: (xbar,_), (n,_), (albedo,rough), (spec,_,_,_)
  float* g_skin_w;     // [n_gauss][B]
  float4* g_quat;      // [n_gauss]
  float4* g_scale_op;  // [n_gauss] (sx,sy,sz,opacity)
  // per-pose
  float4* v_posed;     // [n_verts]
  float4* v_nposed;    // [n_verts]
  float4* g_posed;     // [n_gauss]
  float4* g_nposed;    // [n_gauss]
  float* g_cov;        // [n_gauss][6]
  float* window;       // [4] centre, radius; [4..9] scratch AABB as ordered ints
  unsigned* aabb;      // [8] ordered-uint min xyz, max xyz; [6] counts skin_kernel's finished vertex blocks
  // visibility
  unsigned* rast_sxy;  // [num_sms][n_verts] snapped vertex coordinates of meshes whose table does not fit shared memory
  unsigned* rast_bins; int rast_bins_bands;   // [num_sms][bands][n_faces] triangle lists of banded depth maps (vis_raster)
  unsigned* zmap;      // [max_dirs][res*res]
  int* idmap;          // [max_dirs][res*res]  (allocated lazily at load: always, sized like zmap)
  unsigned* visbits;   // [n_gauss][words]
  unsigned* vbits_a;   // [n_verts][words]
  unsigned* vbits_b;   // [n_verts][words]
  unsigned* vbits_raw; // [n_verts][words]
  unsigned char* vcount;  // [n_verts][max_dirs]
  float* env_table;    // [max_env][8]: w(3), pad, L*A (3), pad
  // shading out
  float4* radiance;    // [n_gauss]
  float4* color;       // [n_gauss]
  float4* attr_color;  // [n_gauss] albedo or posed normal as splat colour (splat_attribute)
  // splat
  float2* mu2d; float* depth; float4* conic_o; int4* rect; unsigned* touched;
  unsigned* tile_count; unsigned* cursor;   // [tiles] histogram of the tile digit, scatter cursors
  unsigned long long* keys[2]; unsigned* vals[2];   // keys[0]: binned local keys (depth<<32|caller index); keys[1]/vals[0]: sorted output (caller indices); vals[1]: the same list as library indices
  unsigned* num_dup;           // [1] D (device)
  uint2* ranges;               // [tiles]
  unsigned* seg_off;           // [tiles + 1] exclusive scan of ceil(n_t / RGA_SEG)
  unsigned* num_items;         // [1] number of (tile, segment) work items (device)
  unsigned* item_tab;          // [items_cap] tile of each work item
  uint2* item_desc;            // [items_cap] (first list entry, tile | entries << 24) of each work item: all the blend needs, in one load
  float4* part;                // [items_cap][256] per-pixel partial (C, T) of each segment
  unsigned* part_last;         // [items_cap][256] last contributing entry of the segment (1-based, 0 = none)
  long long items_cap;
  float* env_pairs;            // [ceil(max_env / 2)][12] environment rows in list order, pairs side by side (fused kernel's table image)
  unsigned* seg_counter;       // [1] item tickets of composite_segment_kernel (zero between launches: the last CTA re-arms it)
  int* stop_seg;               // [pixels] segment in which the pixel's blend stops (-1: list exhausted)
  unsigned char* item_flag;    // [items_cap] work item has pixels to replay (cleared by the replay kernel)
  float* t_final; unsigned* n_contrib;
  double* reg_sums;            // [4] regularisers: sums of Eq.6, 7, 8, 9
  int disp_is_mlp;             // the current displacement is displacement_mlp's v_disp (else the static vt_disp table)
  float* loss_maps; double* loss_sums;   // image_loss: [max_h][max_w][9] SSIM derivative maps, {sum SSIM, sum |I - J|}
  // fused depth test + shading of rga_render_frame (vis_shade_kernels.cu)
  float* frames; int* front_list; unsigned* n_front; unsigned* vs_counter; unsigned* proj_counter; unsigned short* dir_start; unsigned short* tex_list; unsigned short* tex_dir; float* dir_eps;
  int vis_partial; const int* vs_t2d; int vs_rows, vs_cols;   // the frame's visibility words hold only the directions its env map could read
  int* work_counter;           // [1] dynamic work distribution of persistent kernels (zeroed before the launch)
  unsigned* shade_counter;     // [1] group tickets of shade_kernel (zero between launches: the last CTA re-arms it)
  float* splat_grad;           // [n_gauss][12] splat_backward: d_colour(3), d_opacity, d_mu(2), d_conic(3), pad
  int* status;                 // sticky device status
  int sorted_buf;              // which of keys[]/vals[] holds the sorted result
  // state of the current pose
  int have_skin, have_vis, have_shade, have_splat, splat_is_attr;
  int vis_mode, vis_dirs, vis_res, vis_words, keep_maps;
  int vis_culled; float vis_cull_cam[3];   // mode-0 bits were computed only for Gaussians facing this camera (rga_render_frame)
  int cam_w, cam_h;
  long long launches;
  // rga_render_frame: the splat preparation (H6-H9) runs on a second stream beside visibility and shading
  cudaStream_t side;
  cudaEvent_t ev_fork, ev_gskin, ev_env, ev_join;
  // optional per-kernel timing (rga_profile_enable): an event after every kernel, one at every API entry
  int prof_on, prof_n;
  cudaEvent_t prof_ev[RGA_MAX_PROF];
  const char* prof_name[RGA_MAX_PROF];
};
void rga_prof_mark(rga_avatar* av, const char* name, cudaStream_t s);

// ---- launchers (each returns cudaGetLastError()) ----
// load_kernels.cu
cudaError_t rga_launch_knn(const float* q, int nq, const float* v, int nv, int K, int* idx, float* d2, cudaStream_t s);
cudaError_t rga_launch_load_verts(rga_avatar* av, const float* pos, const float* disp, const float* nrm, cudaStream_t s);
cudaError_t rga_launch_load_gauss(rga_avatar* av, const float* gauss_pos, const float* gauss_quat, const float* gauss_scale,
                                  const float* gauss_opacity, const float* d2, cudaStream_t s, const float* vert_quat = nullptr,
                                  const float* vert_scale = nullptr, int set_opacity = 0);
// order_kernels.cu
cudaError_t rga_points_aabb(const float* pos, int n, unsigned* scratch6, float* out6_dev, cudaStream_t s);
cudaError_t rga_build_gauss_order(const float* pos, int n, unsigned long long* keys, int npad, unsigned* bb_u, float* bb_dev,
                                  int* order, int* inv, cudaStream_t s);
cudaError_t rga_gather_rows(int n, int words_per_row, const void* src, const int* order, void* dst, cudaStream_t s);
cudaError_t rga_scatter_rows(int n, int words_per_row, const void* src, const int* order, void* dst, cudaStream_t s);
// skin_kernels.cu
cudaError_t rga_launch_skin(rga_avatar* av, const float* bone_mats, int which, cudaStream_t s);
// vis_kernels.cu
cudaError_t rga_launch_vis_raster(rga_avatar* av, const rga_vis_params* p, cudaStream_t s);
cudaError_t rga_launch_vis_depth_test(rga_avatar* av, const rga_vis_params* p, const float* cull_cam, cudaStream_t s);
cudaError_t rga_launch_vis_paper(rga_avatar* av, const rga_vis_params* p, cudaStream_t s);
size_t rga_vis_raster_smem(int res, int with_id, int n_verts, int* band_rows, int* threads);
int rga_vis_raster_max_bands(int max_res, int n_verts);
int rga_vis_raster_needs_global_table(int max_res, int n_verts);
size_t rga_vis_raster_plan(int res, int with_id, int n_verts, int* band_rows, int* threads, int* sxy_global);
cudaError_t rga_launch_pack_faces(rga_avatar* av, cudaStream_t s);
cudaError_t rga_launch_vertex_normals(const float* x, const int* faces, int nv, int nf, float* out, cudaStream_t s);
// vis_shade_kernels.cu
int rga_vis_shade_teams(int K, int ne);
int rga_vis_shade_init_attributes();
cudaError_t rga_launch_light_frames(rga_avatar* av, const rga_vis_params* p, cudaStream_t s);
cudaError_t rga_launch_front_compact(rga_avatar* av, int words, float3 cam, cudaStream_t s);
cudaError_t rga_launch_texel_csr(rga_avatar* av, const rga_env* env, const rga_vis_params* vis, cudaStream_t s);
cudaError_t rga_launch_vis_shade(rga_avatar* av, const rga_vis_params* vis, const rga_env* env, float3 cam, cudaStream_t s);
// shade_kernels.cu
cudaError_t rga_launch_env_table(rga_avatar* av, const rga_env* env, cudaStream_t s);
cudaError_t rga_launch_shade(rga_avatar* av, const rga_env* env, float3 cam, int vis_mode, cudaStream_t s);
// splat_kernels.cu
cudaError_t rga_launch_project(rga_avatar* av, const rga_camera* cam, cudaStream_t s);
cudaError_t rga_launch_bin(rga_avatar* av, int TX, int ntiles, cudaStream_t s);
cudaError_t rga_launch_tile_sort(rga_avatar* av, const rga_camera* cam, cudaStream_t s);
cudaError_t rga_launch_composite(rga_avatar* av, const rga_camera* cam, float3 bg, const float4* color, float* out, cudaStream_t s);
cudaError_t rga_launch_attr_color(rga_avatar* av, int which, cudaStream_t s);
int rga_init_kernel_attributes();
// mlp_kernels.cu / load_kernels.cu
cudaError_t rga_launch_disp_mlp(rga_avatar* av, const rga_disp_mlp* m, const float* theta, cudaStream_t s);
cudaError_t rga_launch_disp_apply(rga_avatar* av, cudaStream_t s);
cudaError_t rga_launch_disp_static(rga_avatar* av, cudaStream_t s);
cudaError_t rga_build_knn_grid(rga_avatar* av, const float* aabb_host, cudaStream_t s);
cudaError_t rga_launch_knn_gauss(rga_avatar* av, const float* q, cudaStream_t s);
cudaError_t rga_launch_knn_verts(rga_avatar* av, float* d2, cudaStream_t s);
int rga_mlp_init_attributes();
// backward_kernels.cu
cudaError_t rga_launch_splat_backward(rga_avatar* av, const rga_camera* cam, float3 bg, const float* image, const float* dL_dimage,
                                      float* out_dcolor, float* out_dopacity, float* out_dmean, float* out_dcov, cudaStream_t s);
// shade_backward_kernels.cu
cudaError_t rga_launch_shade_backward(rga_avatar* av, const rga_env* env, float3 cam, int vis_mode, const float* dL_dcolor, float* out_dalbedo,
                                      float* out_drough, float* out_dspec, float* out_dnormal, float* out_dpos, float* out_denv, cudaStream_t s);
int rga_shade_backward_init_attributes(int max_env);
// loss_kernels.cu
cudaError_t rga_launch_image_loss_static(const float* image, const float* target, int W, int H, float lam, float* out_loss,
                                         float* out_dimage, cudaStream_t s);
cudaError_t rga_launch_image_loss(rga_avatar* av, const float* image, const float* target, int W, int H, float lam, float* out_loss,
                                  float* out_dimage, cudaStream_t s);
cudaError_t rga_launch_regularisers(rga_avatar* av, float s0, float* out_losses, float* d_alb, float* d_rough, float* d_spec, float* d_gpos,
                                    float* d_disp, float* d_scale, cudaStream_t s);
// pose_backward_kernels.cu
cudaError_t rga_launch_pose_backward(rga_avatar* av, const float* bone_mats, const rga_posed_grads* in, const rga_canonical_grads* out, cudaStream_t s);
// densify_kernels.cu
cudaError_t rga_launch_densify(rga_avatar* av, float d0, float p0, const unsigned* rnd, int max_out, float* out_pos, int* out_tri,
                               int* out_count, cudaStream_t s);
