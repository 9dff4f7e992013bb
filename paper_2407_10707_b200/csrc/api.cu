// C ABI of librga (include/rga.h): argument checks, scratch ownership, stage ordering.  All compute is in the kernels.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <nvtx3/nvToolsExt.h>

// NVTX range per C-ABI call (header-only NVTX 3: a no-op unless a profiler injects itself), so that an Nsight timeline shows
// the path's stages by name (tracing)
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};

#include "rga_internal.h"

int rga_shade_init_attributes(int max_env);
int rga_shade_backward_max_texels();
int rga_vis_init_attributes();
int rga_composite_init_attributes();
int rga_mlp_init_attributes();

static thread_local char g_err[512] = "";
static rga_status fail(rga_status st, const char* fmt, ...) {
  va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap);
  // a CUDA error this call ran into has been reported: do not leave it for the next call's cudaGetLastError to trip over
  if (st == RGA_ERR_CUDA || st == RGA_ERR_OOM) (void)cudaGetLastError();
  return st;
}
#define CU(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return fail(e_ == cudaErrorMemoryAllocation ? RGA_ERR_OOM : RGA_ERR_CUDA, \
    "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)

extern "C" const char* rga_last_error(void) { return g_err; }
extern "C" const char* rga_version(void) { return "rga 0.1 (sm_100a)"; }
extern "C" int64_t rga_launch_count(const rga_avatar* av) { return av ? av->launches : 0; }

void rga_prof_mark(rga_avatar* av, const char* name, cudaStream_t s) {
  if (!av->prof_on || av->prof_n >= RGA_MAX_PROF) return;
  if (!av->prof_ev[av->prof_n]) cudaEventCreate(&av->prof_ev[av->prof_n]);
  cudaEventRecord(av->prof_ev[av->prof_n], s);
  av->prof_name[av->prof_n++] = name;
}

extern "C" rga_status rga_profile_enable(rga_avatar* av, int on) {
  if (!av) return fail(RGA_ERR_INVALID_ARG, "rga_profile_enable: null avatar");
  av->prof_on = on; av->prof_n = 0;
  return RGA_OK;
}

extern "C" rga_status rga_profile_read(rga_avatar* av, void* stream, char* names, float* ms, int capacity, int* count) {
  if (!av || !names || !ms || !count) return fail(RGA_ERR_INVALID_ARG, "rga_profile_read: null argument");
  CU(cudaStreamSynchronize((cudaStream_t)stream));
  int n = 0;
  if (av->prof_on == 2) CU(cudaStreamSynchronize(av->side));
  for (int i = 1; i < av->prof_n && n < capacity; ++i) {
    if (av->prof_name[i][0] == '-') continue;                      // API-entry boundary marks carry no kernel
    float t = 0.f;
    // mode 2 (timeline): both streams stay in use and every mark reports its completion time since the call's entry mark
    CU(cudaEventElapsedTime(&t, av->prof_ev[av->prof_on == 2 ? 0 : i - 1], av->prof_ev[i]));
    snprintf(names + 32 * n, 32, "%s", av->prof_name[i]);
    ms[n++] = t;
  }
  *count = n; av->prof_n = 0;
  return RGA_OK;
}

template <class T> static cudaError_t dalloc(T** p, size_t n) { return cudaMalloc((void**)p, (n ? n : 1) * sizeof(T)); }

extern "C" rga_status avatar_free(rga_avatar* av) {
  if (!av) return RGA_OK;
  void* ptrs[] = {av->vt_quat, av->vt_scale, av->rast_sxy, av->rast_bins, av->frames, av->front_list, av->n_front, av->vs_counter, av->proj_counter, av->dir_start, av->tex_list, av->tex_dir, av->dir_eps, av->g_order, av->g_inv, av->gi_pos, av->bb_scratch, av->bb_dev, av->vals[1], av->reg_sums, av->loss_maps, av->loss_sums, av->work_counter, av->shade_counter, av->splat_grad, av->dens_dv, av->dens_pfix, av->dens_cdf, av->dens_ng, av->dens_block, av->dens_hdr, av->v_pos, av->v_disp, av->g_pos, av->mlp_bias1, av->vt_pos, av->vt_disp, av->vt_normal, av->vt_albedo, av->vt_rough,
                  av->vt_spec, av->knn_d2, av->grid_start, av->grid_verts, av->v_xbar, av->v_normal, av->v_skin_w, av->faces, av->faces_packed, av->knn_v, av->knn_g, av->ubar_g, av->g_static, av->g_skin_w,
                  av->g_quat, av->g_scale_op, av->v_posed, av->v_nposed, av->g_posed, av->g_nposed, av->g_cov, av->window, av->aabb,
                  av->zmap, av->idmap, av->visbits, av->vbits_a, av->vbits_b, av->vbits_raw, av->vcount, av->env_table,
                  av->radiance, av->color, av->attr_color, av->mu2d, av->depth, av->conic_o, av->rect, av->touched, av->tile_count, av->cursor, av->keys[0],
                  av->keys[1], av->vals[0], av->num_dup, av->ranges, av->t_final, av->n_contrib, av->seg_off, av->num_items, av->item_tab, av->part, av->part_last, av->stop_seg, av->item_flag, av->item_desc, av->seg_counter, av->env_pairs,
                  av->status};
  for (void* p : ptrs) if (p) cudaFree(p);
  for (int i = 0; i < RGA_MAX_PROF; ++i) if (av->prof_ev[i]) cudaEventDestroy(av->prof_ev[i]);
  if (av->side) cudaStreamDestroy(av->side);
  if (av->ev_fork) cudaEventDestroy(av->ev_fork);
  if (av->ev_env) cudaEventDestroy(av->ev_env);
  if (av->ev_gskin) cudaEventDestroy(av->ev_gskin);
  if (av->ev_join) cudaEventDestroy(av->ev_join);
  delete av;
  return RGA_OK;
}

extern "C" rga_status avatar_load(const rga_avatar_desc* d, void* stream, rga_avatar** out) {
  NvtxRange nvtx_("rga::avatar_load");
  if (out) *out = nullptr;
  if (!d || !out) return fail(RGA_ERR_INVALID_ARG, "avatar_load: null argument");
  if (d->n_verts < 1 || d->n_faces < 1 || d->n_bones < 1 || d->n_gauss < 1) return fail(RGA_ERR_INVALID_ARG, "avatar_load: empty avatar");
  if (d->k_g < 1 || d->k_g > 3) return fail(RGA_ERR_INVALID_ARG, "avatar_load: k_g must be 1..3");
  if (d->k_v < 1 || d->k_v > 31 || !(d->k_v & 1)) return fail(RGA_ERR_INVALID_ARG, "avatar_load: k_v must be odd, 1..31");
  if (!d->vert_pos || !d->faces || !d->vert_skin_w || !d->vert_albedo || !d->vert_rough || !d->vert_spec ||
      !d->gauss_pos || (!d->gauss_quat && !d->vert_quat) || (!d->gauss_scale && !d->vert_scale))
    return fail(RGA_ERR_INVALID_ARG, "avatar_load: missing table (rotation and scale are needed per Gaussian or per vertex)");
  if (d->max_width < 1 || d->max_height < 1 || d->max_vis_dirs < 1 || d->max_vis_res < 1 || d->max_vis_res > 256 ||
      d->max_env_texels < 1) return fail(RGA_ERR_INVALID_ARG, "avatar_load: bad maxima");
  if ((size_t)d->max_env_texels * 34 + 8 * 1024 > 227 * 1024)
    return fail(RGA_ERR_INVALID_ARG, "avatar_load: max_env_texels = %d is above %d: the shading kernels stage the whole environment table "
                "(34 bytes per texel) in shared memory", d->max_env_texels, (int)((227 * 1024 - 8 * 1024) / 34));
  if (d->n_verts >= (1 << 21)) return fail(RGA_ERR_INVALID_ARG, "avatar_load: n_verts must be below 2^21 (packed faces)");
  if (d->n_faces >= (1 << 24)) return fail(RGA_ERR_INVALID_ARG, "avatar_load: n_faces must be below 2^24 (rasteriser queue entries)");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(RGA_ERR_CUDA, "avatar_load: no CUDA device (there is no CPU fallback)");
  cudaStream_t s = (cudaStream_t)stream;
  rga_avatar* av = new (std::nothrow) rga_avatar();
  if (!av) return fail(RGA_ERR_OOM, "avatar_load: host allocation");
  memset(av, 0, sizeof *av);
  av->n_verts = d->n_verts; av->n_faces = d->n_faces; av->n_bones = d->n_bones; av->n_gauss = d->n_gauss;
  av->k_g = d->k_g; av->k_v = d->k_v;
  if (av->k_v > d->n_verts) av->k_v = (d->n_verts & 1) ? d->n_verts : d->n_verts - 1;      // largest odd count available
  av->max_w = d->max_width; av->max_h = d->max_height; av->max_dirs = d->max_vis_dirs; av->max_res = d->max_vis_res;
  av->max_env = d->max_env_texels;
  av->max_dup = d->max_duplicates > 0 ? d->max_duplicates : (long long)d->n_gauss * 8 + (1 << 18);
  if (av->max_dup > 0xfffffff0ll) av->max_dup = 0xfffffff0ll;
  int dev = 0; cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&av->num_sms, cudaDevAttrMultiProcessorCount, dev);
  const size_t nv = av->n_verts, ng = av->n_gauss, B = av->n_bones, words = (av->max_dirs + 31) / 32;
  const size_t ntiles = (size_t)((av->max_w + 15) / 16) * ((av->max_h + 15) / 16), npix = (size_t)av->max_w * av->max_h;
  const size_t nmap = (size_t)av->max_dirs * av->max_res * av->max_res;
  rga_status st = RGA_OK;
  float* d2 = nullptr;
#define A(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { st = fail(e_ == cudaErrorMemoryAllocation ? RGA_ERR_OOM : RGA_ERR_CUDA, \
    "avatar_load: %s: %s", #call, cudaGetErrorString(e_)); goto done; } } while (0)
  A(dalloc(&av->reg_sums, 4)); A(dalloc(&av->loss_maps, 9 * npix)); A(dalloc(&av->loss_sums, 2)); A(dalloc(&av->work_counter, 1)); A(dalloc(&av->shade_counter, 1)); A(cudaMemsetAsync(av->shade_counter, 0, sizeof(unsigned), s)); A(dalloc(&av->splat_grad, 12 * ng)); A(dalloc(&av->dens_dv, nv)); A(dalloc(&av->dens_pfix, (size_t)av->n_faces)); A(dalloc(&av->dens_cdf, (size_t)av->n_faces));
  A(dalloc(&av->dens_ng, (size_t)av->n_faces)); A(dalloc(&av->dens_block, (size_t)av->n_faces / 2048 + 1)); A(dalloc(&av->dens_hdr, 2));
  A(dalloc(&av->v_pos, nv)); A(dalloc(&av->v_disp, nv)); A(dalloc(&av->g_pos, ng)); A(dalloc(&av->mlp_bias1, 256));
  A(dalloc(&av->v_xbar, nv)); A(dalloc(&av->v_normal, nv)); A(dalloc(&av->v_skin_w, nv * B)); A(dalloc(&av->faces, 3 * (size_t)av->n_faces)); A(dalloc(&av->faces_packed, (size_t)av->n_faces));
  A(dalloc(&av->knn_v, nv * av->k_v)); A(dalloc(&av->knn_g, ng * av->k_g)); A(dalloc(&av->ubar_g, ng * av->k_g));
  A(dalloc(&av->g_static, 4 * ng)); A(dalloc(&av->g_skin_w, ng * B)); A(dalloc(&av->g_quat, ng)); A(dalloc(&av->g_scale_op, ng));
  A(dalloc(&av->v_posed, nv)); A(dalloc(&av->v_nposed, nv)); A(dalloc(&av->g_posed, ng)); A(dalloc(&av->g_nposed, ng));
  A(dalloc(&av->g_cov, 6 * ng)); A(dalloc(&av->window, 4)); A(dalloc(&av->aabb, 8));
  if (rga_vis_raster_needs_global_table(av->max_res, av->n_verts)) A(dalloc(&av->rast_sxy, (size_t)av->num_sms * nv));
  av->rast_bins_bands = rga_vis_raster_max_bands(av->max_res, av->n_verts);
  if (av->rast_bins_bands > 0) A(dalloc(&av->rast_bins, (size_t)av->num_sms * av->rast_bins_bands * (size_t)av->n_faces));
  A(dalloc(&av->zmap, nmap)); A(dalloc(&av->idmap, nmap)); A(dalloc(&av->visbits, ng * words));
  A(dalloc(&av->vbits_a, nv * words)); A(dalloc(&av->vbits_b, nv * words)); A(dalloc(&av->vbits_raw, nv * words));
  A(dalloc(&av->vcount, nv * (size_t)av->max_dirs + 32)); A(dalloc(&av->env_table, 8 * (size_t)av->max_env));
  A(dalloc(&av->radiance, ng)); A(dalloc(&av->color, ng)); A(dalloc(&av->attr_color, ng));
  A(dalloc(&av->mu2d, ng)); A(dalloc(&av->depth, ng)); A(dalloc(&av->conic_o, ng)); A(dalloc(&av->rect, ng)); A(dalloc(&av->touched, ng));
  A(dalloc(&av->tile_count, ntiles)); A(dalloc(&av->cursor, ntiles));
  A(dalloc(&av->keys[0], (size_t)av->max_dup)); A(dalloc(&av->keys[1], (size_t)av->max_dup));
  A(dalloc(&av->vals[0], (size_t)av->max_dup)); A(dalloc(&av->vals[1], (size_t)av->max_dup));
  A(dalloc(&av->frames, 4 * (2 + 3 * (size_t)av->max_dirs))); A(dalloc(&av->front_list, ng)); A(dalloc(&av->n_front, 1)); A(dalloc(&av->vs_counter, 1)); A(dalloc(&av->proj_counter, 1)); A(cudaMemsetAsync(av->proj_counter, 0, sizeof(unsigned), s));
  A(cudaMemsetAsync(av->vs_counter, 0, sizeof(unsigned), s)); A(dalloc(&av->dir_start, (size_t)av->max_dirs + 2)); A(dalloc(&av->tex_list, (size_t)av->max_env + 1)); A(dalloc(&av->tex_dir, (size_t)av->max_env + 1)); A(dalloc(&av->dir_eps, (size_t)av->max_dirs));
  A(dalloc(&av->g_order, ng)); A(dalloc(&av->g_inv, ng)); A(dalloc(&av->gi_pos, 3 * ng)); A(dalloc(&av->bb_scratch, 8)); A(dalloc(&av->bb_dev, 8));
  A(dalloc(&av->num_dup, 1)); A(dalloc(&av->ranges, ntiles));
  av->items_cap = av->max_dup / RGA_SEG + (long long)ntiles + 1;
  A(dalloc(&av->seg_off, ntiles + 1)); A(dalloc(&av->num_items, 1)); A(dalloc(&av->item_tab, (size_t)av->items_cap)); A(dalloc(&av->item_desc, (size_t)av->items_cap));
  A(dalloc(&av->part, (size_t)av->items_cap * 256)); A(dalloc(&av->part_last, (size_t)av->items_cap * 256));
  A(dalloc(&av->env_pairs, 12 * (((size_t)av->max_env + 1) / 2) + 4));
  A(dalloc(&av->seg_counter, 1)); A(cudaMemsetAsync(av->seg_counter, 0, sizeof(unsigned), s));
  A(dalloc(&av->stop_seg, npix)); A(dalloc(&av->item_flag, (size_t)av->items_cap));
  A(cudaMemsetAsync(av->item_flag, 0, (size_t)av->items_cap, s));
  A(dalloc(&av->t_final, npix)); A(dalloc(&av->n_contrib, npix)); A(dalloc(&av->status, 1));
  {
    // the second stream of rga_render_frame carries small, latency-bound kernels: highest priority, so that its CTAs are
    // placed as soon as a CTA of the big kernels on the caller's stream retires
    int prio_lo = 0, prio_hi = 0;
    A(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    A(cudaStreamCreateWithPriority(&av->side, cudaStreamNonBlocking, prio_hi));
  }
  A(cudaEventCreateWithFlags(&av->ev_fork, cudaEventDisableTiming)); A(cudaEventCreateWithFlags(&av->ev_env, cudaEventDisableTiming));
  A(cudaEventCreateWithFlags(&av->ev_gskin, cudaEventDisableTiming));
  A(cudaEventCreateWithFlags(&av->ev_join, cudaEventDisableTiming));
  A(cudaMemsetAsync(av->status, 0, sizeof(int), s)); A(cudaMemsetAsync(av->num_dup, 0, sizeof(unsigned), s));
  {
    unsigned init[8] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u, 0u, 0u};   // [6] = skin_kernel's block counter
    A(cudaMemcpyAsync(av->aabb, init, sizeof init, cudaMemcpyHostToDevice, s));
    A(cudaStreamSynchronize(s));
  }
  A(cudaMemcpyAsync(av->v_skin_w, d->vert_skin_w, nv * B * sizeof(float), cudaMemcpyDeviceToDevice, s));
  A(cudaMemcpyAsync(av->faces, d->faces, 3 * (size_t)av->n_faces * sizeof(int), cudaMemcpyDeviceToDevice, s));
  A(dalloc(&av->vt_pos, 3 * nv)); A(dalloc(&av->vt_normal, 3 * nv)); A(dalloc(&av->vt_albedo, 3 * nv));
  A(dalloc(&av->vt_rough, nv)); A(dalloc(&av->vt_spec, nv)); A(dalloc(&av->knn_d2, ng * av->k_g));
  A(cudaMemcpyAsync(av->vt_pos, d->vert_pos, 3 * nv * sizeof(float), cudaMemcpyDeviceToDevice, s));
  if (d->vert_normal) A(cudaMemcpyAsync(av->vt_normal, d->vert_normal, 3 * nv * sizeof(float), cudaMemcpyDeviceToDevice, s));
  else A(rga_launch_vertex_normals(av->vt_pos, av->faces, av->n_verts, av->n_faces, av->vt_normal, s));   // reading A40
  A(cudaMemcpyAsync(av->vt_albedo, d->vert_albedo, 3 * nv * sizeof(float), cudaMemcpyDeviceToDevice, s));
  A(cudaMemcpyAsync(av->vt_rough, d->vert_rough, nv * sizeof(float), cudaMemcpyDeviceToDevice, s));
  A(cudaMemcpyAsync(av->vt_spec, d->vert_spec, nv * sizeof(float), cudaMemcpyDeviceToDevice, s));
  if (d->vert_quat && !d->gauss_quat) { A(dalloc(&av->vt_quat, 4 * nv)); A(cudaMemcpyAsync(av->vt_quat, d->vert_quat, 4 * nv * sizeof(float), cudaMemcpyDeviceToDevice, s)); }
  if (d->vert_scale && !d->gauss_scale) { A(dalloc(&av->vt_scale, 3 * nv)); A(cudaMemcpyAsync(av->vt_scale, d->vert_scale, 3 * nv * sizeof(float), cudaMemcpyDeviceToDevice, s)); }
  if (d->vert_disp) {
    A(dalloc(&av->vt_disp, 3 * nv));
    A(cudaMemcpyAsync(av->vt_disp, d->vert_disp, 3 * nv * sizeof(float), cudaMemcpyDeviceToDevice, s));
  }
  A(rga_launch_pack_faces(av, s));
  A(rga_launch_load_verts(av, d->vert_pos, d->vert_disp, av->vt_normal, s));
  // KNN: S_v = K_v nearest vertices of each vertex (self included), S_g = K_g nearest of each Gaussian
  A(dalloc(&d2, nv * av->k_v));
  {
    // canonical-vertex AABB for the KNN grid: device reduction, six floats read back (load time)
    float bb[6];
    A(rga_points_aabb(av->vt_pos, av->n_verts, av->bb_scratch, av->bb_dev, s));
    A(cudaMemcpyAsync(bb, av->bb_dev, sizeof bb, cudaMemcpyDeviceToHost, s));
    A(cudaStreamSynchronize(s));
    A(rga_build_knn_grid(av, bb, s));
  }
  A(rga_launch_knn_verts(av, d2, s));
  {
    // Gaussian order (order_kernels.cu): sort once by the Morton code of the canonical position; the caller's per-Gaussian
    // arrays are gathered into library order and every table below is built from those copies
    int npad = 2048; while (npad < av->n_gauss) npad <<= 1;
    unsigned long long* okeys = nullptr; float *pq = nullptr, *ps = nullptr, *po = nullptr;
    cudaError_t e_ = dalloc(&okeys, (size_t)npad);
    if (e_ == cudaSuccess && d->gauss_quat) e_ = dalloc(&pq, 4 * ng);
    if (e_ == cudaSuccess && d->gauss_scale) e_ = dalloc(&ps, 3 * ng);
    if (e_ == cudaSuccess && d->gauss_opacity) e_ = dalloc(&po, ng);
    if (e_ == cudaSuccess) e_ = rga_build_gauss_order(d->gauss_pos, av->n_gauss, okeys, npad, av->bb_scratch, av->bb_dev, av->g_order, av->g_inv, s);
    if (e_ == cudaSuccess) e_ = rga_gather_rows(av->n_gauss, 3, d->gauss_pos, av->g_order, av->gi_pos, s);
    if (e_ == cudaSuccess && pq) e_ = rga_gather_rows(av->n_gauss, 4, d->gauss_quat, av->g_order, pq, s);
    if (e_ == cudaSuccess && ps) e_ = rga_gather_rows(av->n_gauss, 3, d->gauss_scale, av->g_order, ps, s);
    if (e_ == cudaSuccess && po) e_ = rga_gather_rows(av->n_gauss, 1, d->gauss_opacity, av->g_order, po, s);
    if (e_ == cudaSuccess) e_ = rga_launch_knn_gauss(av, av->gi_pos, s);
    if (e_ == cudaSuccess) e_ = rga_launch_load_gauss(av, av->gi_pos, pq, ps, po, av->knn_d2, s, pq ? nullptr : d->vert_quat, ps ? nullptr : d->vert_scale, 1);
    if (e_ == cudaSuccess) e_ = cudaStreamSynchronize(s);
    cudaFree(okeys); cudaFree(pq); cudaFree(ps); cudaFree(po);
    if (e_ != cudaSuccess) { st = fail(e_ == cudaErrorMemoryAllocation ? RGA_ERR_OOM : RGA_ERR_CUDA, "avatar_load: Gaussian order / tables: %s", cudaGetErrorString(e_)); goto done; }
  }
  av->launches += 5;
  if (rga_shade_init_attributes(av->max_env) != 0 || rga_shade_backward_init_attributes(av->max_env) != 0 || rga_vis_init_attributes() != 0 || rga_vis_shade_init_attributes() != 0 || rga_composite_init_attributes() != 0 || rga_mlp_init_attributes() != 0) { st = fail(RGA_ERR_CUDA, "avatar_load: cudaFuncSetAttribute failed"); goto done; }
  A(cudaStreamSynchronize(s));
done:
  if (d2) cudaFree(d2);
  if (st != RGA_OK) { avatar_free(av); return st; }
  *out = av;
  return RGA_OK;
#undef A
}

extern "C" rga_status pose_skin(rga_avatar* av, const float* bone_mats, void* stream) {
  NvtxRange nvtx_("rga::pose_skin");
  if (!av || !bone_mats) return fail(RGA_ERR_INVALID_ARG, "pose_skin: null argument");
  av->have_skin = av->have_vis = av->have_shade = av->have_splat = 0;
  rga_prof_mark(av, "-", (cudaStream_t)stream);
  CU(rga_launch_skin(av, bone_mats, 0, (cudaStream_t)stream));
  av->have_skin = 1;
  return RGA_OK;
}

extern "C" rga_status visibility_raster(rga_avatar* av, const rga_vis_params* p, void* stream) {
  NvtxRange nvtx_("rga::visibility_raster");
  if (!av || !p || !p->dirs) return fail(RGA_ERR_INVALID_ARG, "visibility_raster: null argument");
  if (!av->have_skin) return fail(RGA_ERR_STATE, "visibility_raster: call pose_skin first");
  if (p->n_dirs < 1 || p->n_dirs > av->max_dirs || p->res < 1 || p->res > av->max_res || (p->mode != 0 && p->mode != 1))
    return fail(RGA_ERR_INVALID_ARG, "visibility_raster: n_dirs/res/mode out of range");
  cudaStream_t s = (cudaStream_t)stream;
  av->have_vis = av->have_shade = av->have_splat = 0;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_vis_raster(av, p, s));
  if (p->mode == 0) CU(rga_launch_vis_depth_test(av, p, nullptr, s));
  else CU(rga_launch_vis_paper(av, p, s));
  av->vis_culled = 0; av->vis_partial = 0;
  av->vis_mode = p->mode; av->vis_dirs = p->n_dirs; av->vis_res = p->res; av->vis_words = (p->n_dirs + 31) / 32;
  av->keep_maps = p->keep_maps || p->mode == 1;
  av->have_vis = 1;
  return RGA_OK;
}

extern "C" rga_status shade_gaussians(rga_avatar* av, const rga_env* env, const float cam_pos[3], void* stream) {
  NvtxRange nvtx_("rga::shade_gaussians");
  if (!av || !env || !env->radiance || !cam_pos) return fail(RGA_ERR_INVALID_ARG, "shade_gaussians: null argument");
  if (!av->have_skin) return fail(RGA_ERR_STATE, "shade_gaussians: call pose_skin first");
  if (env->use_visibility && !av->have_vis) return fail(RGA_ERR_STATE, "shade_gaussians: call visibility_raster first");
  if (env->use_visibility && av->vis_mode == 0 && av->vis_culled &&
      (cam_pos[0] != av->vis_cull_cam[0] || cam_pos[1] != av->vis_cull_cam[1] || cam_pos[2] != av->vis_cull_cam[2]))
    return fail(RGA_ERR_STATE, "shade_gaussians: rga_render_frame computed this pose's visibility only for Gaussians facing ITS camera; "
                               "call visibility_raster before shading from another camera");
  if (env->use_visibility && av->vis_mode == 0 && av->vis_partial &&
      ((env->texel_to_dir == nullptr) != (av->vs_t2d == nullptr) || env->rows != av->vs_rows || env->cols != av->vs_cols))
    return fail(RGA_ERR_STATE, "shade_gaussians: rga_render_frame tested only the directions ITS environment map reads; "
                               "call visibility_raster before shading with another map layout");
  if (env->rows < 1 || env->cols < 1 || env->rows * env->cols > av->max_env || !(env->gamma > 0.f))
    return fail(RGA_ERR_INVALID_ARG, "shade_gaussians: env size/gamma out of range");
  if (env->use_visibility && !env->texel_to_dir && env->rows * env->cols != av->vis_dirs)
    return fail(RGA_ERR_INVALID_ARG, "shade_gaussians: identity texel_to_dir needs rows*cols == n_dirs");
  cudaStream_t s = (cudaStream_t)stream;
  av->have_shade = av->have_splat = 0;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_env_table(av, env, s));
  CU(rga_launch_shade(av, env, make_float3(cam_pos[0], cam_pos[1], cam_pos[2]), env->use_visibility ? av->vis_mode : 2, s));
  av->have_shade = 1;
  return RGA_OK;
}

extern "C" rga_status splat_render(rga_avatar* av, const rga_camera* cam, const float bg[3], float* out_image, void* stream) {
  NvtxRange nvtx_("rga::splat_render");
  if (!av || !cam || !bg || !out_image) return fail(RGA_ERR_INVALID_ARG, "splat_render: null argument");
  if (!av->have_shade) return fail(RGA_ERR_STATE, "splat_render: call shade_gaussians first");
  if (cam->width < 1 || cam->height < 1 || cam->width > av->max_w || cam->height > av->max_h)
    return fail(RGA_ERR_INVALID_ARG, "splat_render: camera larger than max_width/max_height");
  cudaStream_t s = (cudaStream_t)stream;
  int TX = (cam->width + 15) / 16, TY = (cam->height + 15) / 16, ntiles = TX * TY;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_project(av, cam, s));
  CU(rga_launch_bin(av, TX, ntiles, s));
  CU(rga_launch_tile_sort(av, cam, s));
  CU(rga_launch_composite(av, cam, make_float3(bg[0], bg[1], bg[2]), av->color, out_image, s));
  av->cam_w = cam->width; av->cam_h = cam->height;
  av->have_splat = 1; av->splat_is_attr = 0;
  return RGA_OK;
}

extern "C" rga_status gaussians_update(rga_avatar* av, const float* gauss_pos, void* stream) {
  NvtxRange nvtx_("rga::gaussians_update");
  if (!av || !gauss_pos) return fail(RGA_ERR_INVALID_ARG, "gaussians_update: null argument");
  cudaStream_t s = (cudaStream_t)stream;
  av->have_skin = av->have_vis = av->have_shade = av->have_splat = 0;
  rga_prof_mark(av, "-", s);
  CU(rga_gather_rows(av->n_gauss, 3, gauss_pos, av->g_order, av->gi_pos, s));      // caller order -> library order (kept from the load)
  CU(rga_launch_knn_gauss(av, av->gi_pos, s));
  rga_prof_mark(av, "knn_g", s);
  CU(rga_launch_load_gauss(av, av->gi_pos, nullptr, nullptr, nullptr, av->knn_d2, s, av->vt_quat, av->vt_scale, 0));
  rga_prof_mark(av, "load_gauss", s);
  av->launches += 3;
  // the displacement network's per-pose dx (if it is the current displacement) is re-interpolated over the new S_g
  if (av->disp_is_mlp) CU(rga_launch_disp_apply(av, s));
  return RGA_OK;
}

extern "C" rga_status splat_backward(rga_avatar* av, const rga_camera* cam, const float bg[3], const float* image, const float* dL_dimage,
                                     float* out_dcolor, float* out_dopacity, float* out_dmean, float* out_dcov, void* stream) {
  NvtxRange nvtx_("rga::splat_backward");
  if (!av || !cam || !bg || !image || !dL_dimage) return fail(RGA_ERR_INVALID_ARG, "splat_backward: null argument");
  if (!av->have_splat || av->splat_is_attr) return fail(RGA_ERR_STATE, "splat_backward: call splat_render (or rga_render_frame) first");
  if (cam->width != av->cam_w || cam->height != av->cam_h) return fail(RGA_ERR_INVALID_ARG, "splat_backward: not the camera of the last splat_render");
  cudaStream_t s = (cudaStream_t)stream;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_splat_backward(av, cam, make_float3(bg[0], bg[1], bg[2]), image, dL_dimage, out_dcolor, out_dopacity, out_dmean, out_dcov, s));
  return RGA_OK;
}

extern "C" rga_status shade_backward(rga_avatar* av, const rga_env* env, const float cam_pos[3], const float* dL_dcolor, float* out_dalbedo,
                                     float* out_drough, float* out_dspec, float* out_dnormal, float* out_dpos, float* out_denv, void* stream) {
  NvtxRange nvtx_("rga::shade_backward");
  if (!av || !env || !env->radiance || !cam_pos || !dL_dcolor) return fail(RGA_ERR_INVALID_ARG, "shade_backward: null argument");
  if (!av->have_shade) return fail(RGA_ERR_STATE, "shade_backward: call shade_gaussians (or rga_render_frame) first");
  if (env->use_visibility && !av->have_vis) return fail(RGA_ERR_STATE, "shade_backward: no visibility for this pose");
  if (env->use_visibility && av->vis_mode == 0 && av->vis_culled &&
      (cam_pos[0] != av->vis_cull_cam[0] || cam_pos[1] != av->vis_cull_cam[1] || cam_pos[2] != av->vis_cull_cam[2]))
    return fail(RGA_ERR_STATE, "shade_backward: this pose's visibility was computed for another camera (rga_render_frame)");
  if (env->use_visibility && av->vis_mode == 0 && av->vis_partial &&
      ((env->texel_to_dir == nullptr) != (av->vs_t2d == nullptr) || env->rows != av->vs_rows || env->cols != av->vs_cols))
    return fail(RGA_ERR_STATE, "shade_backward: this pose's visibility was computed for another environment-map layout (rga_render_frame)");
  if (env->rows < 1 || env->cols < 1 || env->rows * env->cols > av->max_env || !(env->gamma > 0.f))
    return fail(RGA_ERR_INVALID_ARG, "shade_backward: env size/gamma out of range");
  if (env->rows * env->cols > rga_shade_backward_max_texels())
    return fail(RGA_ERR_INVALID_ARG, "shade_backward: %d environment texels are above the %d this kernel can stage in shared memory (46 bytes per "
                "texel; the forward calls take up to %d)", env->rows * env->cols, rga_shade_backward_max_texels(), (int)((227 * 1024 - 8 * 1024) / 34));
  if (env->use_visibility && !env->texel_to_dir && env->rows * env->cols != av->vis_dirs)
    return fail(RGA_ERR_INVALID_ARG, "shade_backward: identity texel_to_dir needs rows*cols == n_dirs");
  cudaStream_t s = (cudaStream_t)stream;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_env_table(av, env, s));
  CU(rga_launch_shade_backward(av, env, make_float3(cam_pos[0], cam_pos[1], cam_pos[2]), env->use_visibility ? av->vis_mode : 2, dL_dcolor,
                               out_dalbedo, out_drough, out_dspec, out_dnormal, out_dpos, out_denv, s));
  return RGA_OK;
}

extern "C" rga_status image_loss(rga_avatar* av, const float* image, const float* target, int width, int height, float lambda,
                                 float* out_loss, float* out_dL_dimage, void* stream) {
  NvtxRange nvtx_("rga::image_loss");
  if (!av || !image || !target) return fail(RGA_ERR_INVALID_ARG, "image_loss: null argument");
  if (width < 1 || height < 1 || width > av->max_w || height > av->max_h) return fail(RGA_ERR_INVALID_ARG, "image_loss: image larger than max_width/max_height");
  if (!(lambda >= 0.f && lambda <= 1.f)) return fail(RGA_ERR_INVALID_ARG, "image_loss: lambda must be in [0, 1]");
  cudaStream_t s = (cudaStream_t)stream;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_image_loss(av, image, target, width, height, lambda, out_loss, out_dL_dimage, s));
  return RGA_OK;
}

extern "C" rga_status rga_image_loss_static(const float* image, const float* target, int width, int height, float lambda,
                                            float* out_loss, float* out_dL_dimage, void* stream) {
  NvtxRange nvtx_("rga::rga_image_loss_static");
  if (!image || !target) return fail(RGA_ERR_INVALID_ARG, "rga_image_loss_static: null argument");
  if (width < 1 || height < 1) return fail(RGA_ERR_INVALID_ARG, "rga_image_loss_static: empty image");
  if ((long long)width * (long long)height > (long long)RGA_IMAGE_LOSS_STATIC_MAX_PIXELS)
    return fail(RGA_ERR_INVALID_ARG, "rga_image_loss_static: %d x %d = %lld pixels is above the static scratch of %d pixels "
                "(RGA_IMAGE_LOSS_STATIC_MAX_PIXELS); use image_loss with an avatar handle for larger images",
                width, height, (long long)width * height, (int)RGA_IMAGE_LOSS_STATIC_MAX_PIXELS);
  if (!(lambda >= 0.f && lambda <= 1.f)) return fail(RGA_ERR_INVALID_ARG, "rga_image_loss_static: lambda must be in [0, 1]");
  CU(rga_launch_image_loss_static(image, target, width, height, lambda, out_loss, out_dL_dimage, (cudaStream_t)stream));
  return RGA_OK;
}

extern "C" rga_status regularisers(rga_avatar* av, float s0, float* out_losses, float* out_dalbedo, float* out_drough, float* out_dspec,
                                   float* out_dgauss_pos, float* out_ddisp, float* out_dscale, void* stream) {
  NvtxRange nvtx_("rga::regularisers");
  if (!av) return fail(RGA_ERR_INVALID_ARG, "regularisers: null avatar");
  cudaStream_t s = (cudaStream_t)stream;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_regularisers(av, s0, out_losses, out_dalbedo, out_drough, out_dspec, out_dgauss_pos, out_ddisp, out_dscale, s));
  return RGA_OK;
}

extern "C" rga_status pose_backward(rga_avatar* av, const float* bone_mats, const rga_posed_grads* in, const rga_canonical_grads* out,
                                    void* stream) {
  NvtxRange nvtx_("rga::pose_backward");
  if (!av || !bone_mats || !in || !out) return fail(RGA_ERR_INVALID_ARG, "pose_backward: null argument");
  if (av->k_g > 8) return fail(RGA_ERR_INVALID_ARG, "pose_backward: k_g > 8 is not supported");
  cudaStream_t s = (cudaStream_t)stream;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_pose_backward(av, bone_mats, in, out, s));
  return RGA_OK;
}

extern "C" rga_status densify_density(rga_avatar* av, float d0, float p0, const uint32_t* rnd, int max_out, float* out_pos,
                                      int32_t* out_tri, int32_t* out_count, void* stream) {
  NvtxRange nvtx_("rga::densify_density");
  if (!av) return fail(RGA_ERR_INVALID_ARG, "densify_density: null avatar");
  if (!(d0 > 0.0f) || d0 > 32768.0f || !(p0 >= 0.0f)) return fail(RGA_ERR_INVALID_ARG, "densify_density: need 0 < d0 <= 32768 and p0 >= 0");
  if (max_out < 0 || (max_out > 0 && (!rnd || !out_pos))) return fail(RGA_ERR_INVALID_ARG, "densify_density: max_out > 0 needs rnd and out_pos");
  if (av->n_faces < 1) return fail(RGA_ERR_INVALID_ARG, "densify_density: the avatar has no triangles");
  cudaStream_t s = (cudaStream_t)stream;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_densify(av, d0, p0, rnd, max_out, out_pos, out_tri, out_count, s));
  return RGA_OK;
}

extern "C" rga_status displacement_mlp(rga_avatar* av, const rga_disp_mlp* mlp, const float* theta, void* stream) {
  NvtxRange nvtx_("rga::displacement_mlp");
  if (!av || !mlp || !theta || !mlp->rff || !mlp->W1 || !mlp->b1 || !mlp->Wh || !mlp->bh || !mlp->Wo || !mlp->bo)
    return fail(RGA_ERR_INVALID_ARG, "displacement_mlp: null argument");
  if (mlp->n_freq < 16 || mlp->n_freq > 128 || (mlp->n_freq & 15) || mlp->n_pose < 0 || mlp->n_pose > 1024)
    return fail(RGA_ERR_INVALID_ARG, "displacement_mlp: n_freq must be a multiple of 16 in [16,128], n_pose in [0,1024]");
  if (mlp->n_pose & 3) return fail(RGA_ERR_INVALID_ARG, "displacement_mlp: n_pose must be a multiple of 4 (16-byte rows of W1)");
  cudaStream_t s = (cudaStream_t)stream;
  av->have_skin = av->have_vis = av->have_shade = av->have_splat = 0;     // the canonical positions change: skin again
  av->disp_is_mlp = 1;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_disp_mlp(av, mlp, theta, s));
  CU(rga_launch_disp_apply(av, s));
  return RGA_OK;
}

// back to the static per-vertex displacement of avatar_load after displacement_mlp
extern "C" rga_status displacement_static(rga_avatar* av, void* stream) {
  NvtxRange nvtx_("rga::displacement_static");
  if (!av) return fail(RGA_ERR_INVALID_ARG, "displacement_static: null avatar");
  cudaStream_t s = (cudaStream_t)stream;
  av->have_skin = av->have_vis = av->have_shade = av->have_splat = 0;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_disp_static(av, s));
  CU(rga_launch_disp_apply(av, s));
  av->disp_is_mlp = 0;
  return RGA_OK;
}

extern "C" rga_status splat_attribute(rga_avatar* av, const rga_camera* cam, const float bg[3], int which, float* out_image,
                                      void* stream) {
  NvtxRange nvtx_("rga::splat_attribute");
  if (!av || !cam || !bg || !out_image) return fail(RGA_ERR_INVALID_ARG, "splat_attribute: null argument");
  if (which != RGA_ATTR_ALBEDO && which != RGA_ATTR_NORMAL) return fail(RGA_ERR_INVALID_ARG, "splat_attribute: unknown attribute %d", which);
  if (!av->have_skin) return fail(RGA_ERR_STATE, "splat_attribute: call pose_skin first");
  if (cam->width < 1 || cam->height < 1 || cam->width > av->max_w || cam->height > av->max_h)
    return fail(RGA_ERR_INVALID_ARG, "splat_attribute: camera larger than max_width/max_height");
  cudaStream_t s = (cudaStream_t)stream;
  const int TX = (cam->width + 15) / 16, TY = (cam->height + 15) / 16, ntiles = TX * TY;
  rga_prof_mark(av, "-", s);
  CU(rga_launch_attr_color(av, which, s));
  CU(rga_launch_project(av, cam, s));
  CU(rga_launch_bin(av, TX, ntiles, s));
  CU(rga_launch_tile_sort(av, cam, s));
  CU(rga_launch_composite(av, cam, make_float3(bg[0], bg[1], bg[2]), av->attr_color, out_image, s));
  av->cam_w = cam->width; av->cam_h = cam->height;
  av->have_splat = 1; av->splat_is_attr = 1;      // the blend state now belongs to the attribute map, not to the shaded frame
  return RGA_OK;
}

// One whole frame.  Same kernels as the four calls above, but the splat preparation (H6 projection, H7 binning, H8 sort,
// H9 ranges) and the environment table do not depend on visibility or shading, so they run on the avatar's second stream
// beside H3-H5 and join before the blend (fork / join by events: still CUDA-graph-capturable).
extern "C" rga_status rga_render_frame(rga_avatar* av, const float* bone_mats, const rga_vis_params* vis, const rga_env* env,
                                       const float cam_pos[3], const rga_camera* cam, const float bg[3], float* out_image,
                                       void* stream) {
  NvtxRange nvtx_("rga::rga_render_frame");
  if (!av || !bone_mats || !env || !env->radiance || !cam_pos || !cam || !bg || !out_image)
    return fail(RGA_ERR_INVALID_ARG, "rga_render_frame: null argument");
  if (env->use_visibility && !vis) return fail(RGA_ERR_INVALID_ARG, "rga_render_frame: use_visibility needs vis params");
  if (vis && (!vis->dirs || vis->n_dirs < 1 || vis->n_dirs > av->max_dirs || vis->res < 1 || vis->res > av->max_res ||
              (vis->mode != 0 && vis->mode != 1)))
    return fail(RGA_ERR_INVALID_ARG, "rga_render_frame: n_dirs/res/mode out of range");
  if (env->rows < 1 || env->cols < 1 || env->rows * env->cols > av->max_env || !(env->gamma > 0.f))
    return fail(RGA_ERR_INVALID_ARG, "rga_render_frame: env size/gamma out of range");
  if (env->use_visibility && !env->texel_to_dir && env->rows * env->cols != vis->n_dirs)
    return fail(RGA_ERR_INVALID_ARG, "rga_render_frame: identity texel_to_dir needs rows*cols == n_dirs");
  if (cam->width < 1 || cam->height < 1 || cam->width > av->max_w || cam->height > av->max_h)
    return fail(RGA_ERR_INVALID_ARG, "rga_render_frame: camera larger than max_width/max_height");
  cudaStream_t s = (cudaStream_t)stream;
  const bool overlap = av->prof_on != 1;                   // per-kernel events need one stream (mode 2 = timeline keeps both)
  cudaStream_t s2 = overlap ? av->side : s;
  // a failure after the fork must not leave the second stream un-joined (inside a CUDA-graph capture that would invalidate
  // the capture): join it, forget the half-built pose state, then report
  bool forked = false;
#define CUF(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { \
    if (forked) { cudaEventRecord(av->ev_join, s2); cudaStreamWaitEvent(s, av->ev_join, 0); } \
    av->have_skin = av->have_vis = av->have_shade = av->have_splat = 0; \
    return fail(e_ == cudaErrorMemoryAllocation ? RGA_ERR_OOM : RGA_ERR_CUDA, "rga_render_frame: %s: %s", #expr, cudaGetErrorString(e_)); } } while (0)
  const int TX = (cam->width + 15) / 16, TY = (cam->height + 15) / 16, ntiles = TX * TY;
  av->have_skin = av->have_vis = av->have_shade = av->have_splat = 0;
  rga_prof_mark(av, "-", s);
  const float3 cam3 = make_float3(cam_pos[0], cam_pos[1], cam_pos[2]);
  // mode 0 inside one frame: camera, environment map and texel -> direction map are known when visibility is tested, so the
  // depth test and the shading run as ONE kernel over the camera-facing Gaussians (vis_shade_kernels.cu)
  const bool fused = vis && vis->mode == 0 && env->use_visibility && rga_vis_shade_teams(vis->n_dirs, env->rows * env->cols) > 0;
  if (overlap) {
    // the rasteriser only needs the posed mesh and the window: the Gaussians are skinned on the second stream
    CUF(cudaEventRecord(av->ev_fork, s)); CUF(cudaStreamWaitEvent(s2, av->ev_fork, 0)); forked = true;
    CUF(rga_launch_skin(av, bone_mats, 1, s));
    CUF(rga_launch_skin(av, bone_mats, 2, s2));
  } else CUF(rga_launch_skin(av, bone_mats, 0, s));
  av->have_skin = 1;
  if (fused) CUF(rga_launch_front_compact(av, (vis->n_dirs + 31) / 32, cam3, s2));
  if (overlap) CUF(cudaEventRecord(av->ev_gskin, s2));
  CUF(rga_launch_env_table(av, env, s2));
  if (fused) CUF(rga_launch_texel_csr(av, env, vis, s2));
  if (overlap) CUF(cudaEventRecord(av->ev_env, s2));
  CUF(rga_launch_project(av, cam, s2));
  CUF(rga_launch_bin(av, TX, ntiles, s2));
  CUF(rga_launch_tile_sort(av, cam, s2));
  if (overlap) CUF(cudaEventRecord(av->ev_join, s2));
  av->vis_partial = 0;
  if (vis) {
    CUF(rga_launch_vis_raster(av, vis, s));
    if (overlap) CUF(cudaStreamWaitEvent(s, av->ev_gskin, 0));
    if (fused) {
      if (overlap) CUF(cudaStreamWaitEvent(s, av->ev_env, 0));
      CUF(rga_launch_vis_shade(av, vis, env, cam3, s));
      av->vis_culled = 1; av->vis_cull_cam[0] = cam_pos[0]; av->vis_cull_cam[1] = cam_pos[1]; av->vis_cull_cam[2] = cam_pos[2];
      av->vis_partial = 1; av->vs_t2d = env->texel_to_dir; av->vs_rows = env->rows; av->vs_cols = env->cols;
    } else if (vis->mode == 0) {
      CUF(rga_launch_vis_depth_test(av, vis, cam_pos, s));
      av->vis_culled = 1; av->vis_cull_cam[0] = cam_pos[0]; av->vis_cull_cam[1] = cam_pos[1]; av->vis_cull_cam[2] = cam_pos[2];
    } else {
      CUF(rga_launch_vis_paper(av, vis, s));
      av->vis_culled = 0;
    }
    av->vis_mode = vis->mode; av->vis_dirs = vis->n_dirs; av->vis_res = vis->res; av->vis_words = (vis->n_dirs + 31) / 32;
    av->keep_maps = vis->keep_maps || vis->mode == 1;
    av->have_vis = 1;
  }
  if (!fused) {
    if (overlap) { if (!vis) CUF(cudaStreamWaitEvent(s, av->ev_gskin, 0)); CUF(cudaStreamWaitEvent(s, av->ev_env, 0)); }
    CUF(rga_launch_shade(av, env, cam3, env->use_visibility ? av->vis_mode : 2, s));
  }
  av->have_shade = 1;
  if (overlap) CUF(cudaStreamWaitEvent(s, av->ev_join, 0));
  CUF(rga_launch_composite(av, cam, make_float3(bg[0], bg[1], bg[2]), av->color, out_image, s));
  av->cam_w = cam->width; av->cam_h = cam->height;
  av->have_splat = 1; av->splat_is_attr = 0;
  return RGA_OK;
#undef CUF
}

extern "C" rga_status rga_check(rga_avatar* av, void* stream) {
  if (!av) return fail(RGA_ERR_INVALID_ARG, "rga_check: null avatar");
  int st = 0;
  CU(cudaMemcpyAsync(&st, av->status, sizeof st, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CU(cudaStreamSynchronize((cudaStream_t)stream));
  if (st != 0) { cudaMemsetAsync(av->status, 0, sizeof(int), (cudaStream_t)stream); return fail((rga_status)st, "device status %d (capacity overflow: raise max_duplicates)", st); }
  return RGA_OK;
}

extern "C" rga_status rga_get_buffer(rga_avatar* av, int which, void* stream, const void** dev_ptr, size_t* bytes) {
  if (!av || !dev_ptr || !bytes) return fail(RGA_ERR_INVALID_ARG, "rga_get_buffer: null argument");
  const size_t nv = av->n_verts, ng = av->n_gauss, words = av->vis_words, K = av->vis_dirs, R = av->vis_res;
  const size_t npix = (size_t)av->cam_w * av->cam_h, ntiles = (size_t)((av->cam_w + 15) / 16) * ((av->cam_h + 15) / 16);
  size_t D = 0;
  if (which == RGA_BUF_KEYS_SORTED || which == RGA_BUF_VALS_SORTED) {
    unsigned d = 0;
    CU(cudaMemcpyAsync(&d, av->num_dup, 4, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    D = d; if ((long long)D > av->max_dup) D = (size_t)av->max_dup;
  }
  const void* p = nullptr; size_t n = 0;
  switch (which) {
    case RGA_BUF_KNN_G: p = av->knn_g; n = ng * av->k_g * 4; break;
    case RGA_BUF_UBAR_G: p = av->ubar_g; n = ng * av->k_g * 4; break;
    case RGA_BUF_KNN_V: p = av->knn_v; n = nv * av->k_v * 4; break;
    case RGA_BUF_GAUSS_STATIC: p = av->g_static; n = ng * 64; break;
    case RGA_BUF_GAUSS_SKIN_W: p = av->g_skin_w; n = ng * av->n_bones * 4; break;
    case RGA_BUF_VERT_POSED: p = av->v_posed; n = nv * 16; break;
    case RGA_BUF_VERT_NORMAL_POSED: p = av->v_nposed; n = nv * 16; break;
    case RGA_BUF_GAUSS_POSED: p = av->g_posed; n = ng * 16; break;
    case RGA_BUF_GAUSS_NORMAL_POSED: p = av->g_nposed; n = ng * 16; break;
    case RGA_BUF_GAUSS_COV: p = av->g_cov; n = ng * 24; break;
    case RGA_BUF_WINDOW: p = av->window; n = 16; break;
    case RGA_BUF_ZMAP: p = av->zmap; n = K * R * R * 4; break;
    case RGA_BUF_IDMAP: p = av->idmap; n = av->keep_maps ? K * R * R * 4 : 0; break;
    case RGA_BUF_VISBITS: p = av->visbits; n = ng * words * 4; break;
    case RGA_BUF_VCOUNT: p = av->vcount; n = nv * K; break;
    case RGA_BUF_RADIANCE: p = av->radiance; n = ng * 16; break;
    case RGA_BUF_COLOR: p = av->color; n = ng * 16; break;
    case RGA_BUF_MU2D: p = av->mu2d; n = ng * 8; break;
    case RGA_BUF_DEPTH: p = av->depth; n = ng * 4; break;
    case RGA_BUF_CONIC_OPACITY: p = av->conic_o; n = ng * 16; break;
    case RGA_BUF_RECT: p = av->rect; n = ng * 16; break;
    case RGA_BUF_TOUCHED: p = av->touched; n = ng * 4; break;
    case RGA_BUF_NUM_DUPLICATES: p = av->num_dup; n = 4; break;
    case RGA_BUF_KEYS_SORTED: p = av->keys[1]; n = D * 8; break;
    case RGA_BUF_VALS_SORTED: p = av->vals[0]; n = D * 4; break;
    case RGA_BUF_TILE_RANGES: p = av->ranges; n = ntiles * 8; break;
    case RGA_BUF_T_FINAL: p = av->t_final; n = npix * 4; break;
    case RGA_BUF_N_CONTRIB: p = av->n_contrib; n = npix * 4; break;
    case RGA_BUF_VERT_BITS_RAW: p = av->vbits_raw; n = nv * words * 4; break;
    case RGA_BUF_VERT_DISP: p = av->v_disp; n = nv * 16; break;
    case RGA_BUF_SPLAT_GRAD: p = av->splat_grad; n = ng * 48; break;
    case RGA_BUF_DENS_DV: p = av->dens_dv; n = nv * 4; break;
    case RGA_BUF_DENS_P: p = av->dens_pfix; n = (size_t)av->n_faces * 4; break;
    case RGA_BUF_DENS_NG: p = av->dens_ng; n = (size_t)av->n_faces * 4; break;
    case RGA_BUF_DENS_HDR: p = av->dens_hdr; n = 16; break;
    case RGA_BUF_GAUSS_ORDER: p = av->g_order; n = ng * 4; break;
    case RGA_BUF_VERT_NORMAL: p = av->vt_normal; n = nv * 12; break;
    default: return fail(RGA_ERR_INVALID_ARG, "rga_get_buffer: unknown id %d", which);
  }
  *dev_ptr = p; *bytes = n;
  return RGA_OK;
}

static bool per_gaussian_buffer(int which) {
  switch (which) {
    case RGA_BUF_KNN_G: case RGA_BUF_UBAR_G: case RGA_BUF_GAUSS_STATIC: case RGA_BUF_GAUSS_SKIN_W: case RGA_BUF_GAUSS_POSED:
    case RGA_BUF_GAUSS_NORMAL_POSED: case RGA_BUF_GAUSS_COV: case RGA_BUF_VISBITS: case RGA_BUF_RADIANCE: case RGA_BUF_COLOR:
    case RGA_BUF_MU2D: case RGA_BUF_DEPTH: case RGA_BUF_CONIC_OPACITY: case RGA_BUF_RECT: case RGA_BUF_TOUCHED: case RGA_BUF_SPLAT_GRAD:
      return true;
    default: return false;
  }
}

extern "C" rga_status rga_read_buffer(rga_avatar* av, int which, void* stream, void* host_dst, size_t capacity, size_t* bytes) {
  const void* p = nullptr; size_t n = 0;
  rga_status st = rga_get_buffer(av, which, stream, &p, &n);
  if (st != RGA_OK) return st;
  if (bytes) *bytes = n;
  if (!host_dst || capacity < n) return fail(RGA_ERR_INVALID_ARG, "rga_read_buffer: need %zu bytes", n);
  cudaStream_t s = (cudaStream_t)stream;
  if (n && per_gaussian_buffer(which)) {
    // per-Gaussian tables live in the library's spatial order: rows are put back into the CALLER's order on the way out
    void* tmp = nullptr;
    CU(cudaMalloc(&tmp, n));
    cudaError_t e = rga_scatter_rows(av->n_gauss, (int)(n / 4 / (size_t)av->n_gauss), p, av->g_order, tmp, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(host_dst, tmp, n, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(tmp);
    if (e != cudaSuccess) return fail(RGA_ERR_CUDA, "rga_read_buffer: %s", cudaGetErrorString(e));
    return RGA_OK;
  }
  if (n) CU(cudaMemcpyAsync(host_dst, p, n, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  return RGA_OK;
}
