// ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain, slow, scalar CPU restatement of the per-frame forward render of
// arXiv 2407.10707.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may call it.  It shares no code with the CUDA path (paper_2407_10707_b200/csrc) and neither includes the other.
//
// Precision: every quantity that decides an integer output (KNN order, tile
// rects, sort keys, depth maps, visibility bits) is computed in fp32 with the operation order written here and NO
// IMPLICIT fused multiply-add (build with -ffp-contract=off); only + - * / sqrt and, where written, an explicit
// std::fma -- all of which IEEE-754 rounds identically on every machine.  Everything compared under a tolerance (shading, compositing) is computed in double.
//
// Pins (tests/test_oracle_pins.py, tests/test_oracle_pins2.py): see DESIGN.md "Oracle pins".  "parity unpinned" only for
// the VALUES of: gamma exponent (A9), shadow-map bias constants (A17), 3DGS rasteriser constants (A18) -- PAPER.md prints
// no value for them; the RULES that use them (clamp, skip, stop-before, n_contrib; bias monotone in the slope) are pinned.
// Arithmetic frozen since round 2 (reading A37): a kernel that wants another operation order matches this file.
//
// Build: g++ -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC (oracle/build.py).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#define ORC extern "C" __attribute__((visibility("default")))

static inline float dot3(const float* a, const float* b) { return (a[0] * b[0] + a[1] * b[1]) + a[2] * b[2]; }
static inline float dot3(float ax, float ay, float az, float bx, float by, float bz) { return (ax * bx + ay * by) + az * bz; }
static inline uint32_t fbits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
static inline float bitsf(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }

// ---------------------------------------------------------------------------------------------------------------
// L0  K nearest canonical-mesh vertices (PAPER.md:93 S_g, :120 S_v, :193 K_g=3 K_v=19).  Brute force IS the
// definition.  d2 = (dx*dx + dy*dy) + dz*dz in fp32; K smallest; ties -> lower vertex index; ascending.
ORC void orc_knn(const float* q, int nq, const float* v, int nv, int K, int32_t* idx, float* d2out) {
#pragma omp parallel for schedule(static)
  for (int i = 0; i < nq; ++i) {
    std::vector<float> bd(K, INFINITY);
    std::vector<int32_t> bi(K, -1);
    for (int j = 0; j < nv; ++j) {
      float dx = q[3 * i] - v[3 * j], dy = q[3 * i + 1] - v[3 * j + 1], dz = q[3 * i + 2] - v[3 * j + 2];
      float d = (dx * dx + dy * dy) + dz * dz;
      if (d < bd[K - 1]) {                       // strict: an equal distance never displaces a lower index
        int p = K - 1;
        while (p > 0 && d < bd[p - 1]) { bd[p] = bd[p - 1]; bi[p] = bi[p - 1]; --p; }
        bd[p] = d; bi[p] = j;
      }
    }
    for (int k = 0; k < K; ++k) { idx[(size_t)i * K + k] = bi[k]; d2out[(size_t)i * K + k] = bd[k]; }
  }
}

// Eq.1 weights: u_j = 1/||x_g - x_j||_2, normalised so they sum to 1 (reading A1: clamp at 1e-12).
ORC void orc_interp_weights(const float* d2, int n, int K, float* ubar) {
  for (int i = 0; i < n; ++i) {
    float U = 0.0f;
    std::vector<float> u(K);
    for (int k = 0; k < K; ++k) {
      float dist = std::sqrt(d2[(size_t)i * K + k]);
      u[k] = 1.0f / std::fmax(dist, 1e-12f);
      U = (k == 0) ? u[0] : U + u[k];
    }
    for (int k = 0; k < K; ++k) ubar[(size_t)i * K + k] = u[k] / U;
  }
}

// Eq.1: *_g = sum_j ubar_j *_j, accumulated in neighbour order j = 0..K-1, fp32, no FMA.
ORC void orc_interp_attr(const int32_t* idx, const float* ubar, int n, int K, const float* attr, int C, float* out) {
  for (int i = 0; i < n; ++i)
    for (int c = 0; c < C; ++c) {
      float acc = ubar[(size_t)i * K] * attr[(size_t)idx[(size_t)i * K] * C + c];
      for (int k = 1; k < K; ++k) acc = acc + ubar[(size_t)i * K + k] * attr[(size_t)idx[(size_t)i * K + k] * C + c];
      out[(size_t)i * C + c] = acc;
    }
}

// Eq.1 for the rotation attribute r (reading A2): q and -q are the same rotation, so every neighbour's
// quaternion first takes the sign of neighbour 0's (dot4 < 0 -> negated); then the weighted sum in neighbour order, fp32,
// no FMA.  The result is NOT normalised here: orc_gauss_cov normalises the quaternion it is given.
ORC void orc_interp_quat(const int32_t* idx, const float* ubar, int n, int K, const float* vq, float* out) {
  for (int i = 0; i < n; ++i) {
    const float* q0 = vq + 4 * (size_t)idx[(size_t)i * K];
    float acc[4];
    for (int c = 0; c < 4; ++c) acc[c] = ubar[(size_t)i * K] * q0[c];
    for (int k = 1; k < K; ++k) {
      const float* qk = vq + 4 * (size_t)idx[(size_t)i * K + k];
      float dt = ((qk[0] * q0[0] + qk[1] * q0[1]) + qk[2] * q0[2]) + qk[3] * q0[3];
      float sg = dt < 0.0f ? -1.0f : 1.0f;
      for (int c = 0; c < 4; ++c) acc[c] = acc[c] + ubar[(size_t)i * K + k] * (sg * qk[c]);
    }
    for (int c = 0; c < 4; ++c) out[4 * (size_t)i + c] = acc[c];
  }
}

ORC void orc_normalize_rows3(float* v, int n) {
  for (int i = 0; i < n; ++i) {
    float* p = v + 3 * (size_t)i;
    float len = std::sqrt(dot3(p, p));
    if (len > 0.0f) { p[0] = p[0] / len; p[1] = p[1] / len; p[2] = p[2] / len; }
  }
}

// L0, vertex normals when the caller stores nothing but geometry (PAPER.md:86 lists n among the vertex attributes and does
// not say where it comes from; NULL = area-weighted normals of the canonical mesh; reading A40).
// n_v = normalize( sum over the faces f = 0..nf-1 in ascending order, corners k = 0..2, that touch v, of
// (x_b - x_a) x (x_c - x_a) ): the cross product's length is twice the face area, so the sum is area-weighted.  fp32, one
// rounding per operation, in this order (the normal decides visibility bits downstream); a vertex without a face keeps 0.
ORC void orc_vertex_normals(const float* x, const int* faces, int nv, int nf, float* out) {
  for (size_t i = 0; i < 3 * (size_t)nv; ++i) out[i] = 0.0f;
  for (int f = 0; f < nf; ++f) {
    const int* t = faces + 3 * (size_t)f;
    const float *a = x + 3 * (size_t)t[0], *b = x + 3 * (size_t)t[1], *c = x + 3 * (size_t)t[2];
    float e1[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]}, e2[3] = {c[0] - a[0], c[1] - a[1], c[2] - a[2]};
    float cr[3] = {e1[1] * e2[2] - e1[2] * e2[1], e1[2] * e2[0] - e1[0] * e2[2], e1[0] * e2[1] - e1[1] * e2[0]};
    for (int k = 0; k < 3; ++k) {
      float* o = out + 3 * (size_t)t[k];
      o[0] = o[0] + cr[0]; o[1] = o[1] + cr[1]; o[2] = o[2] + cr[2];
    }
  }
  orc_normalize_rows3(out, nv);
}

// ---------------------------------------------------------------------------------------------------------------
// H1/H2 forward LBS (reading A3).  M = sum_b w_b G_b accumulated b = 0..B-1 from +0;
// x' = M [x + dx; 1];  n' = normalize(M3x3 n).  Also returns M (12 floats per point) for the covariance step.
ORC void orc_skin(const float* x, const float* dx, const float* nrm, const float* w, int n, int B, const float* G,
                  float* xo, float* no, float* Mo) {
#pragma omp parallel for schedule(static)
  for (int i = 0; i < n; ++i) {
    float M[12];
    for (int e = 0; e < 12; ++e) M[e] = 0.0f;
    for (int b = 0; b < B; ++b) {
      float wb = w[(size_t)i * B + b];
      for (int e = 0; e < 12; ++e) M[e] = M[e] + wb * G[b * 12 + e];
    }
    float p[3];
    for (int c = 0; c < 3; ++c) p[c] = x[3 * (size_t)i + c] + (dx ? dx[3 * (size_t)i + c] : 0.0f);
    for (int r = 0; r < 3; ++r)
      xo[3 * (size_t)i + r] = ((M[4 * r] * p[0] + M[4 * r + 1] * p[1]) + M[4 * r + 2] * p[2]) + M[4 * r + 3];
    float t[3];
    const float* nn = nrm + 3 * (size_t)i;
    for (int r = 0; r < 3; ++r) t[r] = (M[4 * r] * nn[0] + M[4 * r + 1] * nn[1]) + M[4 * r + 2] * nn[2];
    float len = std::sqrt(dot3(t, t));
    for (int r = 0; r < 3; ++r) no[3 * (size_t)i + r] = (len > 0.0f) ? t[r] / len : t[r];
    if (Mo) for (int e = 0; e < 12; ++e) Mo[12 * (size_t)i + e] = M[e];
  }
}

// H2 covariance (PAPER.md:95 "rotation ... rotated accordingly", :103; reading A3): Sigma = A A^T,
// A = M3x3 R(q) diag(s), q = (w,x,y,z) normalised first.  Output xx,xy,xz,yy,yz,zz.
ORC void orc_gauss_cov(const float* M, const float* q, const float* s, int n, float* cov6) {
  for (int i = 0; i < n; ++i) {
    const float* qq = q + 4 * (size_t)i;
    float ql = std::sqrt(((qq[0] * qq[0] + qq[1] * qq[1]) + qq[2] * qq[2]) + qq[3] * qq[3]);
    float w = qq[0] / ql, x = qq[1] / ql, y = qq[2] / ql, z = qq[3] / ql;
    float R[9] = {1.0f - 2.0f * (y * y + z * z), 2.0f * (x * y - w * z), 2.0f * (x * z + w * y),
                  2.0f * (x * y + w * z), 1.0f - 2.0f * (x * x + z * z), 2.0f * (y * z - w * x),
                  2.0f * (x * z - w * y), 2.0f * (y * z + w * x), 1.0f - 2.0f * (x * x + y * y)};
    float RS[9], A[9];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) RS[3 * r + c] = R[3 * r + c] * s[3 * (size_t)i + c];
    const float* Mi = M + 12 * (size_t)i;
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c)
      A[3 * r + c] = (Mi[4 * r] * RS[c] + Mi[4 * r + 1] * RS[3 + c]) + Mi[4 * r + 2] * RS[6 + c];
    float* o = cov6 + 6 * (size_t)i;
    int k = 0;
    for (int r = 0; r < 3; ++r) for (int c = r; c < 3; ++c)
      o[k++] = (A[3 * r] * A[3 * c] + A[3 * r + 1] * A[3 * c + 1]) + A[3 * r + 2] * A[3 * c + 2];
  }
}

// Orthographic window shared by all light directions (reading A13): bounding sphere of the posed-vertex AABB.
ORC void orc_window(const float* x, int n, float* c3, float* r) {
  float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c) {
    mn[c] = std::fmin(mn[c], x[3 * (size_t)i + c]); mx[c] = std::fmax(mx[c], x[3 * (size_t)i + c]);
  }
  float dg[3];
  for (int c = 0; c < 3; ++c) { c3[c] = (mn[c] + mx[c]) * 0.5f; dg[c] = mx[c] - mn[c]; }
  float rr = (0.5f * std::sqrt(dot3(dg, dg))) * 1.015625f;
  *r = (rr > 0.0f) ? rr : 1.0f;
}

// Light frame (reading A13): w = direction toward the light; u = normalize(e x w), e = z unless |w_z| > 0.999; v = w x u.
static void light_frame(const float* w, float* u, float* v) {
  float e[3] = {0.0f, 0.0f, 1.0f};
  if (std::fabs(w[2]) > 0.999f) { e[0] = 1.0f; e[2] = 0.0f; }
  float c[3] = {e[1] * w[2] - e[2] * w[1], e[2] * w[0] - e[0] * w[2], e[0] * w[1] - e[1] * w[0]};
  float len = std::sqrt(dot3(c, c));
  for (int k = 0; k < 3; ++k) u[k] = c[k] / len;
  v[0] = w[1] * u[2] - w[2] * u[1]; v[1] = w[2] * u[0] - w[0] * u[2]; v[2] = w[0] * u[1] - w[1] * u[0];
}
ORC void orc_light_frames(const float* dirs, int K, float* uvw) {
  for (int k = 0; k < K; ++k) {
    light_frame(dirs + 3 * k, uvw + 9 * k, uvw + 9 * k + 3);
    for (int c = 0; c < 3; ++c) uvw[9 * k + 6 + c] = dirs[3 * k + c];
  }
}

// Light-space projection of one point (reading A13): continuous pixel coords (px,py) and normalised depth z
// (0 = nearest the light).  Per direction the frame is pre-scaled once, u_s = u sR, v_s = v sR, w_n = -w inv2r with
// sR = (R/2)/r, hR = R/2, inv2r = 1/(2r); per point the work is three fused multiply-add chains on d = p - c:
//   px = fma(u_s.z, d.z, fma(u_s.y, d.y, fma(u_s.x, d.x, hR)))      = (u.d) sR + R/2
//   py = likewise with v_s
//   z  = fma(w_n.z, d.z, fma(w_n.y, d.y, fma(w_n.x, d.x, 0.5)))     = (r - w.d) / (2r)
// std::fma is the correctly rounded fused operation on every IEEE-754 machine, so this stays bit-reproducible.
// DIAGNOSTIC ONLY (reading A37): the same projection and bias in the spelled-out form of SURVEY.md:371-381,
//   px = ((u.d)/r * 1/2 + 1/2) R,  z = (r - w.d)/(2r),  beta = ((bias_texels (2r/R)) tau + bias_world)/(2r),
// selected by orc_set_plain_projection(1).  oracle/a37_projection_forms.py counts the depth texels and visibility bits
// that differ between the two forms; nothing else ever switches it on.
static int g_plain_projection = 0;
ORC void orc_set_plain_projection(int on) { g_plain_projection = on; }

static inline void light_project(const float* p, const float* c, float r, const float* u, const float* v, const float* w,
                                 int R, float* px, float* py, float* z) {
  if (g_plain_projection) {
    float d[3] = {p[0] - c[0], p[1] - c[1], p[2] - c[2]};
    *px = ((dot3(u, d) / r) * 0.5f + 0.5f) * (float)R;
    *py = ((dot3(v, d) / r) * 0.5f + 0.5f) * (float)R;
    *z = (r - dot3(w, d)) / (2.0f * r);
    return;
  }
  float hR = 0.5f * (float)R, sR = hR / r, inv2r = 1.0f / (2.0f * r);
  float us[3] = {u[0] * sR, u[1] * sR, u[2] * sR}, vs[3] = {v[0] * sR, v[1] * sR, v[2] * sR};
  float wn[3] = {-(w[0] * inv2r), -(w[1] * inv2r), -(w[2] * inv2r)};
  float d[3] = {p[0] - c[0], p[1] - c[1], p[2] - c[2]};
  *px = std::fma(us[2], d[2], std::fma(us[1], d[1], std::fma(us[0], d[0], hR)));
  *py = std::fma(vs[2], d[2], std::fma(vs[1], d[1], std::fma(vs[0], d[0], hR)));
  *z = std::fma(wn[2], d[2], std::fma(wn[1], d[1], std::fma(wn[0], d[0], 0.5f)));
}

// ---------------------------------------------------------------------------------------------------------------
// H3 visibility rasterisation ("orthographic projection towards the 512 directions and rasterize the
// projected triangles ... each pixel of which indicates the rasterized triangle index").  Conventions: readings
// A13/A14 and SURVEY 8(c) step 4.  Vertices snapped to 1/256 pixel (round-half-even), int64 edge functions, pixel
// centre covered when the three edge functions share a sign or are zero (two-sided, inclusive), depth
// z = (z0 + (e1/area)(z1-z0)) + (e2/area)(z2-z0) in fp32, clamped at 0, winner = min (zbits << 32 | tri).
// zmap: [K][R][R] float bits, 0xFFFFFFFF = empty; idmap: [K][R][R] triangle id, -1 = empty (may be NULL).
// cull != 0 (reading A36, an option for closed, outward-oriented meshes): a triangle whose snapped area is negative --
// it faces away from the light -- is skipped like a zero-area one.
ORC void orc_vis_raster(const float* xp, int nv, const int32_t* f, int nf, const float* dirs, int K, int R,
                        const float* c, float r, uint32_t* zmap, int32_t* idmap, int cull) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int k = 0; k < K; ++k) {
    float u[3], v[3]; const float* w = dirs + 3 * k;
    light_frame(w, u, v);
    std::vector<int32_t> X(nv), Y(nv); std::vector<float> Z(nv);
    for (int i = 0; i < nv; ++i) {
      float px, py, z; light_project(xp + 3 * (size_t)i, c, r, u, v, w, R, &px, &py, &z);
      X[i] = (int32_t)std::nearbyint(px * 256.0f); Y[i] = (int32_t)std::nearbyint(py * 256.0f); Z[i] = z;
    }
    std::vector<uint64_t> best((size_t)R * R, ~0ull);
    for (int t = 0; t < nf; ++t) {
      int i0 = f[3 * t], i1 = f[3 * t + 1], i2 = f[3 * t + 2];
      int64_t x0 = X[i0], y0 = Y[i0], x1 = X[i1], y1 = Y[i1], x2 = X[i2], y2 = Y[i2];
      int64_t area = (x1 - x0) * (y2 - y0) - (y1 - y0) * (x2 - x0);
      if (area == 0) continue;
      if (cull && area < 0) continue;
      int64_t mnx = std::min(x0, std::min(x1, x2)), mxx = std::max(x0, std::max(x1, x2));
      int64_t mny = std::min(y0, std::min(y1, y2)), mxy = std::max(y0, std::max(y1, y2));
      // pixel i has centre 256 i + 128: first i with centre >= mnx, last with centre <= mxx
      int64_t ia = (mnx - 128 + 255) >> 8, ib = (mxx - 128) >> 8, ja = (mny - 128 + 255) >> 8, jb = (mxy - 128) >> 8;
      ia = std::max<int64_t>(ia, 0); ja = std::max<int64_t>(ja, 0);
      ib = std::min<int64_t>(ib, R - 1); jb = std::min<int64_t>(jb, R - 1);
      float z0 = Z[i0], z1 = Z[i1], z2 = Z[i2], fa = (float)area;
      for (int64_t j = ja; j <= jb; ++j) for (int64_t i = ia; i <= ib; ++i) {
        int64_t qx = 256 * i + 128, qy = 256 * j + 128;
        int64_t e0 = (x2 - x1) * (qy - y1) - (y2 - y1) * (qx - x1);
        int64_t e1 = (x0 - x2) * (qy - y2) - (y0 - y2) * (qx - x2);
        int64_t e2 = (x1 - x0) * (qy - y0) - (y1 - y0) * (qx - x0);
        bool in = (e0 >= 0 && e1 >= 0 && e2 >= 0) || (e0 <= 0 && e1 <= 0 && e2 <= 0);
        if (!in) continue;
        float t1 = (float)e1 / fa, t2 = (float)e2 / fa;
        float z = (z0 + t1 * (z1 - z0)) + t2 * (z2 - z0);
        z = std::fmax(z, 0.0f);
        uint64_t key = ((uint64_t)fbits(z) << 32) | (uint32_t)t;
        uint64_t& b = best[(size_t)j * R + i];
        if (key < b) b = key;
      }
    }
    for (size_t p = 0; p < (size_t)R * R; ++p) {
      zmap[(size_t)k * R * R + p] = (uint32_t)(best[p] >> 32);
      if (idmap) idmap[(size_t)k * R * R + p] = (best[p] == ~0ull) ? -1 : (int32_t)(best[p] & 0xFFFFFFFFu);
    }
  }
}

// H4a shadow-map depth test (BASELINE.json north_star (b); PAPER.md:124 names it as the contrast case; reading A17).
// bits: [ng][K/32 words]; bit (k%32) of word k/32 of row g is 1 when Gaussian g sees direction k.
ORC void orc_vis_depth_test(const float* xg, const float* ng_, int ng, const float* dirs, int K, int R, const float* c,
                            float r, const uint32_t* zmap, float bias_texels, float bias_world, float slope_max,
                            uint32_t* bits) {
  int words = (K + 31) / 32;
  std::memset(bits, 0, (size_t)ng * words * 4);
  std::vector<float> U(3 * K), V(3 * K);
  for (int k = 0; k < K; ++k) light_frame(dirs + 3 * k, &U[3 * k], &V[3 * k]);
#pragma omp parallel for schedule(static)
  for (int g = 0; g < ng; ++g) {
    for (int k = 0; k < K; ++k) {
      const float* w = dirs + 3 * k;
      float px, py, z; light_project(xg + 3 * (size_t)g, c, r, &U[3 * k], &V[3 * k], w, R, &px, &py, &z);
      float fxp = std::fmin(std::fmax(std::floor(px), 0.0f), (float)(R - 1));
      float fyp = std::fmin(std::fmax(std::floor(py), 0.0f), (float)(R - 1));
      int ix = (int)fxp, iy = (int)fyp;
      uint32_t zb = zmap[((size_t)k * R + iy) * R + ix];
      bool vis;
      if (zb == 0xFFFFFFFFu) vis = true;
      else {
        float cs = dot3(ng_ + 3 * (size_t)g, w), tau;
        if (cs > 0.0f) {
          float s2 = std::fmax(1.0f - cs * cs, 0.0f);
          tau = std::sqrt(s2) / cs;
          tau = std::fmin(std::fmax(tau, 1.0f), slope_max);
        } else tau = slope_max;
        float beta = (bias_texels / (float)R) * tau + bias_world * (1.0f / (2.0f * r));   // texel = 1/R in normalised depth
        if (g_plain_projection) beta = ((bias_texels * ((2.0f * r) / (float)R)) * tau + bias_world) / (2.0f * r);
        vis = z <= bitsf(zb) + beta;
      }
      if (vis) bits[(size_t)g * words + (k >> 5)] |= 1u << (k & 31);
    }
  }
}

// H4b paper visibility (Eq.3 :113, Eq.4 :118; readings A14-A16).
// raw[k][j] = 1 if any triangle containing vertex j wins >= 1 pixel in map k; median = majority of the Kv bits at
// S_v (self included, Kv odd); twice; mean = count of ones among S_v -> vcount[j][k] in 0..Kv  (vertex-major u8).
// raw_out / med1_out / med2_out ([K][nv] u8, may be NULL) expose the intermediate maps.
ORC void orc_vis_paper(const int32_t* idmap, const int32_t* f, int nf, int nv, int K, int R, const int32_t* knn_v,
                       int Kv, uint8_t* vcount, uint8_t* raw_out, uint8_t* med1_out, uint8_t* med2_out) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int k = 0; k < K; ++k) {
    std::vector<uint8_t> a(nv, 0), b(nv, 0);
    for (size_t p = 0; p < (size_t)R * R; ++p) {
      int32_t t = idmap[(size_t)k * R * R + p];
      if (t >= 0) { a[f[3 * t]] = 1; a[f[3 * t + 1]] = 1; a[f[3 * t + 2]] = 1; }
    }
    if (raw_out) std::memcpy(raw_out + (size_t)k * nv, a.data(), nv);
    for (int pass = 0; pass < 2; ++pass) {
      for (int j = 0; j < nv; ++j) {
        int s = 0;
        for (int q = 0; q < Kv; ++q) s += a[knn_v[(size_t)j * Kv + q]];
        b[j] = (2 * s > Kv) ? 1 : 0;              // median of Kv (odd) bits
      }
      a.swap(b);
      if (pass == 0 && med1_out) std::memcpy(med1_out + (size_t)k * nv, a.data(), nv);
      if (pass == 1 && med2_out) std::memcpy(med2_out + (size_t)k * nv, a.data(), nv);
    }
    for (int j = 0; j < nv; ++j) {
      int s = 0;
      for (int q = 0; q < Kv; ++q) s += a[knn_v[(size_t)j * Kv + q]];
      vcount[(size_t)j * K + k] = (uint8_t)s;
    }
  }
}

// Gaussian visibility attribute (Eq.1 applied to v): v_g[k] = sum_j ubar_j vbar_j[k], vbar = count/Kv.
ORC void orc_vis_gauss(const uint8_t* vcount, const int32_t* knn_g, const float* ubar, int ng, int Kg, int K, int Kv,
                       double* vg) {
#pragma omp parallel for schedule(static)
  for (int g = 0; g < ng; ++g)
    for (int k = 0; k < K; ++k) {
      double acc = 0.0;
      for (int q = 0; q < Kg; ++q)
        acc += (double)ubar[(size_t)g * Kg + q] * ((double)vcount[(size_t)knn_g[(size_t)g * Kg + q] * K + k] / (double)Kv);
      vg[(size_t)g * K + k] = acc;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Environment quadrature ("light probes L in R^{16x32x3} with 512 discrete area lights"; reading A6):
// equirectangular z-up, texel (i,j): theta=(i+1/2)pi/R, phi=(j+1/2)2pi/C, w toward the light,
// A = (cos(i pi/R) - cos((i+1) pi/R)) 2pi/C  (exact solid angle; sum = 4 pi).
ORC void orc_env_table(int rows, int cols, double* w3, double* A) {
  const double PI = 3.14159265358979323846;
  for (int i = 0; i < rows; ++i) for (int j = 0; j < cols; ++j) {
    double th = (i + 0.5) * PI / rows, ph = (j + 0.5) * 2.0 * PI / cols;
    size_t k = (size_t)i * cols + j;
    w3[3 * k] = std::sin(th) * std::cos(ph); w3[3 * k + 1] = std::sin(th) * std::sin(ph); w3[3 * k + 2] = std::cos(th);
    A[k] = (std::cos(i * PI / rows) - std::cos((i + 1) * PI / rows)) * 2.0 * PI / cols;
  }
}

// BRDF, Appendix A, Eq.12-15 verbatim, with Eq.12's G/(4 (n.wi)(n.wo)) evaluated in the
// algebraically identical cancelled form 1/(4 ((n.wi)(1-k)+k) ((n.wo)(1-k)+k)) (reading A10).
// Returns R per channel (3).  Caller guarantees n.wi > 0.  n.wo is clamped at 0 (grazing / back-facing view).
static void brdf(const double* wi, const double* wo, const double* n, const double* a, double rough, double spec,
                 double* out) {
  const double PI = 3.14159265358979323846;
  double h[3] = {wi[0] + wo[0], wi[1] + wo[1], wi[2] + wo[2]};
  double hl = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
  double s = 0.0;
  if (hl > 0.0) {
    for (int c = 0; c < 3; ++c) h[c] /= hl;
    double nh = n[0] * h[0] + n[1] * h[1] + n[2] * h[2];
    double oh = wo[0] * h[0] + wo[1] * h[1] + wo[2] * h[2];
    double ni = n[0] * wi[0] + n[1] * wi[1] + n[2] * wi[2];
    double no = std::max(0.0, n[0] * wo[0] + n[1] * wo[1] + n[2] * wo[2]);
    double al = rough * rough, al2 = al * al;                                   // Eq.13: alpha = gamma^2
    double den = nh * nh * (al2 - 1.0) + 1.0;
    double D = al2 / (PI * den * den);
    double F = 0.04 + (1.0 - 0.04) * std::exp2((-5.55473 * oh - 6.98316) * oh); // Eq.14, F0 = 0.04 (:471)
    double k = (rough + 1.0) * (rough + 1.0) / 8.0;                             // Eq.15
    s = D * F / (4.0 * (ni * (1.0 - k) + k) * (no * (1.0 - k) + k));
  }
  for (int c = 0; c < 3; ++c) out[c] = a[c] / PI + spec * s;                     // Eq.12
}
ORC void orc_brdf(const double* wi, const double* wo, const double* n, const double* a, double rough, double spec,
                  double* out) { brdf(wi, wo, n, a, rough, spec, out); }

// H5 shading, Eq.2: L_o = sum_k L^k A^k R(w_i^k, w_o, n) v_g[k] max(0, w_i^k . n); colour =
// clamp(L_o,0,1)^(1/gamma) (reading A9).  w_o = normalize(cam - x) (A7).  vis_mode 0: v_g[k] = bit texel_to_dir[k]
// of bits[g]; 1: v_g[k] = vg[g][texel_to_dir[k]] (double); 2: v = 1.  texel_to_dir NULL = identity.
ORC void orc_shade(const float* xg, const float* ng_, const float* alb, const float* rough, const float* spec, int ng,
                   const float* cam, const float* env, int rows, int cols, const int32_t* t2d, int vis_mode,
                   const uint32_t* bits, const double* vg, int K, double gamma, double* Lo, double* cg) {
  int ne = rows * cols, words = (K + 31) / 32;
  std::vector<double> W(3 * (size_t)ne), A(ne);
  orc_env_table(rows, cols, W.data(), A.data());
#pragma omp parallel for schedule(static)
  for (int g = 0; g < ng; ++g) {
    double x[3], n[3], a[3], wo[3];
    for (int c = 0; c < 3; ++c) { x[c] = xg[3 * (size_t)g + c]; n[c] = ng_[3 * (size_t)g + c]; a[c] = alb[3 * (size_t)g + c]; }
    for (int c = 0; c < 3; ++c) wo[c] = (double)cam[c] - x[c];
    double wl = std::sqrt(wo[0] * wo[0] + wo[1] * wo[1] + wo[2] * wo[2]);
    for (int c = 0; c < 3; ++c) wo[c] /= wl;
    double acc[3] = {0, 0, 0};
    for (int k = 0; k < ne; ++k) {
      const double* wi = &W[3 * (size_t)k];
      double cs = wi[0] * n[0] + wi[1] * n[1] + wi[2] * n[2];
      if (cs <= 0.0) continue;                                   // max(0, w_i . n)
      int d = t2d ? t2d[k] : k;
      double v = 1.0;
      if (vis_mode == 0) v = (bits[(size_t)g * words + (d >> 5)] >> (d & 31)) & 1u ? 1.0 : 0.0;
      else if (vis_mode == 1) v = vg[(size_t)g * K + d];
      if (v == 0.0) continue;
      double Rr[3];
      brdf(wi, wo, n, a, (double)rough[g], (double)spec[g], Rr);
      for (int c = 0; c < 3; ++c) acc[c] += (double)env[3 * (size_t)k + c] * A[k] * Rr[c] * v * cs;
    }
    for (int c = 0; c < 3; ++c) {
      Lo[3 * (size_t)g + c] = acc[c];
      cg[3 * (size_t)g + c] = std::pow(std::min(1.0, std::max(0.0, acc[c])), 1.0 / gamma);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// H6 projection + culling (PAPER.md:101 back-face rule, :103 "the Gaussian rasterizer of 3DGS" -> ref [8]; readings
// A8, A18, A21).  fp32, op order as written, no FMA: this decides tile rects and sort keys.
// cam: R_wc[9] row-major, t_wc[3], fx, fy, cx, cy, width, height, z_near  (15 floats, width/height as floats)
// out: mu[ng][2], depth[ng], conic_o[ng][4] (a,b,c,opacity), rect[ng][4] (x0,y0,x1,y1 tiles, half-open), touched[ng]
ORC void orc_project(const float* xg, const float* ng_, const float* cov6, const float* opac, int ng, const float* cam,
                     float* mu, float* depth, float* conic_o, int32_t* rect, uint32_t* touched, int32_t* radius_out) {
  const float* Rw = cam; const float* tw = cam + 9;
  float fx = cam[12], fy = cam[13], cx = cam[14], cy = cam[15];
  int W = (int)cam[16], H = (int)cam[17]; float znear = cam[18];
  int TX = (W + 15) / 16, TY = (H + 15) / 16;
  float C[3];                                                     // camera centre = -R^T t
  for (int r = 0; r < 3; ++r) C[r] = -((Rw[r] * tw[0] + Rw[3 + r] * tw[1]) + Rw[6 + r] * tw[2]);
  float limx = 1.3f * ((float)W / (2.0f * fx)), limy = 1.3f * ((float)H / (2.0f * fy));
  for (int g = 0; g < ng; ++g) {
    const float* x = xg + 3 * (size_t)g;
    touched[g] = 0;
    for (int c = 0; c < 4; ++c) { rect[4 * (size_t)g + c] = 0; conic_o[4 * (size_t)g + c] = 0.0f; }
    mu[2 * (size_t)g] = mu[2 * (size_t)g + 1] = 0.0f; depth[g] = 0.0f; if (radius_out) radius_out[g] = 0;
    float t[3];
    for (int r = 0; r < 3; ++r) t[r] = ((Rw[3 * r] * x[0] + Rw[3 * r + 1] * x[1]) + Rw[3 * r + 2] * x[2]) + tw[r];
    if (!(t[2] > znear)) continue;
    float wo[3] = {C[0] - x[0], C[1] - x[1], C[2] - x[2]};
    if (dot3(ng_ + 3 * (size_t)g, wo) < 0.0f) continue;          // facing away -> opacity 0
    float txz = std::fmin(limx, std::fmax(-limx, t[0] / t[2])) * t[2];
    float tyz = std::fmin(limy, std::fmax(-limy, t[1] / t[2])) * t[2];
    float J00 = fx / t[2], J02 = -(fx * txz) / (t[2] * t[2]), J11 = fy / t[2], J12 = -(fy * tyz) / (t[2] * t[2]);
    float T0[3], T1[3];
    for (int j = 0; j < 3; ++j) { T0[j] = J00 * Rw[j] + J02 * Rw[6 + j]; T1[j] = J11 * Rw[3 + j] + J12 * Rw[6 + j]; }
    const float* s = cov6 + 6 * (size_t)g;
    float S[9] = {s[0], s[1], s[2], s[1], s[3], s[4], s[2], s[4], s[5]};
    float V0[3], V1[3];
    for (int a = 0; a < 3; ++a) {
      V0[a] = (T0[0] * S[a] + T0[1] * S[3 + a]) + T0[2] * S[6 + a];
      V1[a] = (T1[0] * S[a] + T1[1] * S[3 + a]) + T1[2] * S[6 + a];
    }
    float c00 = dot3(V0, T0) + 0.3f, c01 = dot3(V0, T1), c11 = dot3(V1, T1) + 0.3f;
    float det = c00 * c11 - c01 * c01;
    if (!(det > 0.0f)) continue;
    float mid = 0.5f * (c00 + c11);
    float lam = mid + std::sqrt(std::fmax(0.1f, mid * mid - det));
    float rad = std::ceil(3.0f * std::sqrt(lam));
    float mx = (fx * t[0]) / t[2] + cx, my = (fy * t[1]) / t[2] + cy;
    float x0 = std::fmin(std::fmax(std::floor((mx - rad) / 16.0f), 0.0f), (float)TX);
    float x1 = std::fmin(std::fmax(std::floor(((mx + rad) + 15.0f) / 16.0f), 0.0f), (float)TX);
    float y0 = std::fmin(std::fmax(std::floor((my - rad) / 16.0f), 0.0f), (float)TY);
    float y1 = std::fmin(std::fmax(std::floor(((my + rad) + 15.0f) / 16.0f), 0.0f), (float)TY);
    int ix0 = (int)x0, ix1 = (int)x1, iy0 = (int)y0, iy1 = (int)y1;
    if ((ix1 - ix0) * (iy1 - iy0) <= 0) continue;
    mu[2 * (size_t)g] = mx; mu[2 * (size_t)g + 1] = my; depth[g] = t[2];
    conic_o[4 * (size_t)g] = c11 / det; conic_o[4 * (size_t)g + 1] = -c01 / det; conic_o[4 * (size_t)g + 2] = c00 / det;
    conic_o[4 * (size_t)g + 3] = opac ? opac[g] : 1.0f;
    rect[4 * (size_t)g] = ix0; rect[4 * (size_t)g + 1] = iy0; rect[4 * (size_t)g + 2] = ix1; rect[4 * (size_t)g + 3] = iy1;
    touched[g] = (uint32_t)((ix1 - ix0) * (iy1 - iy0));
    if (radius_out) radius_out[g] = (int32_t)rad;
  }
}

// H7 + H8: emit (tile << 32 | depth bits, g) for every tile of every rect, Gaussians ascending, tiles row-major;
// stable sort by key (reading A22).  Returns D.  keys/vals must hold sum(touched) entries.
ORC int64_t orc_emit_sort(const float* depth, const int32_t* rect, const uint32_t* touched, int ng, int TX,
                          uint64_t* keys, uint32_t* vals) {
  std::vector<std::pair<uint64_t, uint32_t>> kv;
  for (int g = 0; g < ng; ++g) {
    if (!touched[g]) continue;
    const int32_t* r = rect + 4 * (size_t)g;
    for (int y = r[1]; y < r[3]; ++y) for (int x = r[0]; x < r[2]; ++x)
      kv.push_back({((uint64_t)(uint32_t)(y * TX + x) << 32) | fbits(depth[g]), (uint32_t)g});
  }
  std::stable_sort(kv.begin(), kv.end(), [](const auto& a, const auto& b) { return a.first < b.first; });
  for (size_t i = 0; i < kv.size(); ++i) { keys[i] = kv[i].first; vals[i] = kv[i].second; }
  return (int64_t)kv.size();
}

// H9: ranges[t] = [first, last+1) of tile t in the sorted keys; empty tiles get (0,0).
ORC void orc_tile_ranges(const uint64_t* keys, int64_t D, int ntiles, uint32_t* ranges) {
  std::memset(ranges, 0, (size_t)ntiles * 8);
  for (int64_t i = 0; i < D; ++i) {
    uint32_t t = (uint32_t)(keys[i] >> 32);
    if (i == 0 || (uint32_t)(keys[i - 1] >> 32) != t) ranges[2 * t] = (uint32_t)i;
    if (i == D - 1 || (uint32_t)(keys[i + 1] >> 32) != t) ranges[2 * t + 1] = (uint32_t)(i + 1);
  }
}

// One pixel's front-to-back blend over an index list (3DGS conventions, reading A18): double precision.
// flag (test bookkeeping, not part of the method; SURVEY.md:224-227, reading A38): set when one of the three
// threshold decisions lies within the reach of an fp32 evaluation of the same formulas, so that a correct fp32 blend may
// legitimately take the other branch.  The reach is derived from the arithmetic, with U = 2^-23 (one fp32 ulp, relative):
//   power: an fp32 evaluation of -0.5(a dx^2 + c dy^2) - b dx dy carries an absolute error of at most 4 U M, where
//          M = 0.5(|a| dx^2 + |c| dy^2) + |b dx dy| >= |power| is the magnitude of its terms;
//   alpha: o exp(power) inherits that as a relative error, plus 16 U for the exponential (ex2.approx is good to 2 ulp,
//          its argument power * log2(e) is rounded twice) and the product:  rel(alpha) <= (16 + 4 M) U;
//   T:     a product of n fp32 factors (1 - alpha_i) carries the relative error sum_i [U + delta(alpha_i) / (1 - alpha_i)]
//          (an alpha clamped to 0.99 on both sides contributes no delta).
// The flag says WHICH decision can flip, because the three move the pixel by different amounts (reading A38): bit 0 = alpha
// against 1/255 (one contribution of alpha = 1/255), bit 1 = the stopping rule (the entry that takes T to 1e-4 contributes
// alpha T with T (1 - alpha) = 1e-4: up to 0.99 / 0.01 * 1e-4 = 9.9e-3), bit 2 = the sign of power (a whole contribution).
static void blend_pixel(double pxc, double pyc, const uint32_t* list, int64_t n, const float* mu, const float* conic_o,
                        const double* col, const float* bg, double* out3, double* Tout, uint32_t* ncontrib, uint8_t* flag) {
  const double U = 1.1920928955078125e-07;                 // 2^-23
  double T = 1.0, C[3] = {0, 0, 0}, eT = 0.0; uint32_t cnt = 0, last = 0; uint8_t fl = 0;
  for (int64_t i = 0; i < n; ++i) {
    uint32_t g = list[i]; ++cnt;
    double dx = (double)mu[2 * (size_t)g] - pxc, dy = (double)mu[2 * (size_t)g + 1] - pyc;
    const float* co = conic_o + 4 * (size_t)g;
    double power = -0.5 * ((double)co[0] * dx * dx + (double)co[2] * dy * dy) - (double)co[1] * dx * dy;
    double M = 0.5 * (std::fabs((double)co[0]) * dx * dx + std::fabs((double)co[2]) * dy * dy) + std::fabs((double)co[1] * dx * dy);
    if (power != 0.0 && std::fabs(power) <= 8.0 * U * M) fl |= 4;
    if (power > 0.0) continue;
    double raw = (double)co[3] * std::exp(power), rel = (16.0 + 4.0 * M) * U;
    double alpha = std::min(0.99, raw);
    if (std::fabs(alpha - 1.0 / 255.0) <= rel * alpha) fl |= 1;
    if (alpha < 1.0 / 255.0) continue;
    double dalpha = (raw > 0.99 * (1.0 + rel)) ? 0.0 : rel * alpha;       // clamped on both sides: exact
    double testT = T * (1.0 - alpha), eTest = eT + 2.0 * U + dalpha / (1.0 - alpha);
    if (std::fabs(testT - 1e-4) <= eTest * testT) fl |= 2;
    if (testT < 1e-4) break;
    for (int c = 0; c < 3; ++c) C[c] += col[3 * (size_t)g + c] * alpha * T;
    T = testT; eT = eTest; last = cnt;
  }
  for (int c = 0; c < 3; ++c) out3[c] = C[c] + T * (double)bg[c];
  *Tout = T; *ncontrib = last; if (flag) *flag = fl;
}

// H10 tiled compositing: pixel (i,j) samples at (i+1/2, j+1/2) (A21) over its 16x16 tile's sorted list.
ORC void orc_composite(const uint32_t* vals, const uint32_t* ranges, const float* mu, const float* conic_o,
                       const double* col, const float* bg, int W, int H, double* image, double* Tfinal,
                       uint32_t* ncontrib, uint8_t* flags) {
  int TX = (W + 15) / 16;
#pragma omp parallel for schedule(dynamic, 4)
  for (int y = 0; y < H; ++y) for (int x = 0; x < W; ++x) {
    int t = (y / 16) * TX + (x / 16);
    size_t p = (size_t)y * W + x;
    blend_pixel(x + 0.5, y + 0.5, vals + ranges[2 * t], (int64_t)ranges[2 * t + 1] - ranges[2 * t], mu, conic_o, col, bg,
                image + 3 * p, Tfinal + p, ncontrib + p, flags ? flags + p : nullptr);
  }
}

// Per-pixel brute force (north_star invariant): ALL Gaussians with touched>0, ordered by (depth bits, index); one
// contributes to a pixel iff the pixel's tile lies inside its tile rect.  Must equal orc_composite exactly.
ORC void orc_composite_bruteforce(const float* depth, const int32_t* rect, const uint32_t* touched, int ng,
                                  const float* mu, const float* conic_o, const double* col, const float* bg, int W,
                                  int H, double* image, double* Tfinal, uint32_t* ncontrib) {
  std::vector<uint32_t> order;
  for (int g = 0; g < ng; ++g) if (touched[g]) order.push_back((uint32_t)g);
  std::stable_sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) { return fbits(depth[a]) < fbits(depth[b]); });
#pragma omp parallel for schedule(dynamic, 4)
  for (int y = 0; y < H; ++y) {
    std::vector<uint32_t> list;
    for (int x = 0; x < W; ++x) {
      int tx = x / 16, ty = y / 16;
      list.clear();
      for (uint32_t g : order) {
        const int32_t* r = rect + 4 * (size_t)g;
        if (tx >= r[0] && tx < r[2] && ty >= r[1] && ty < r[3]) list.push_back(g);
      }
      size_t p = (size_t)y * W + x;
      blend_pixel(x + 0.5, y + 0.5, list.data(), (int64_t)list.size(), mu, conic_o, col, bg, image + 3 * p, Tfinal + p,
                  ncontrib + p, nullptr);
    }
  }
}
