// Target evaluation on the device: x -> (f, p, pixel, score)  (rows a3-a6).
//   a3 raygen / extend, a4 BVH8 closest hit (software; top levels in shared memory), a5 shade,
//   a6 score = grad p / (p + eps) by reverse accumulation over the recorded vertices.
// The path map is DESIGN.md Q4-Q9 (the paper does not describe its path sampling routines).
#pragma once
#include <cfloat>
#include <cstdint>
#include <cuda_runtime.h>

#include "dr_types.h"

namespace dr {

constexpr float kEps = 1e-8f;
constexpr float kTwoPi = 6.283185307179586f;
constexpr int kStackDepth = 64;

struct DevScene {
  const float4* nodes;  // Node8 as 16 float4
  const float4* tris;   // TriPacked as 3 float4
  const float4* mats;   // MatPacked as 3 float4
  uint32_t n_nodes, smem_nodes, n_tris, n_mats;
  float env[3];
  float cam_pos[3], cam_w[3], cam_r[3], cam_v[3];
  float tan_half, tan_half_aspect;
  uint32_t W, H, L, d, planes;
  float eps_ray;
  int analytic, n_mix;
  float mix_w[kMaxMix], mix_mx[kMaxMix], mix_my[kMaxMix], mix_s[kMaxMix];
};

// ---- small vector helpers -----------------------------------------------------------------------------
__device__ __forceinline__ float3 operator+(float3 a, float3 b) { return make_float3(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ float3 operator-(float3 a, float3 b) { return make_float3(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ float3 operator*(float3 a, float s) { return make_float3(a.x * s, a.y * s, a.z * s); }
__device__ __forceinline__ float dot3(float3 a, float3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ float3 cross3(float3 a, float3 b) {
  return make_float3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
__device__ __forceinline__ float3 normalize3(float3 a) { return a * (1.0f / sqrtf(dot3(a, a))); }
__device__ __forceinline__ float3 xyz(float4 q) { return make_float3(q.x, q.y, q.z); }

// ---- forward-mode numbers with K tangents (local Jacobians of one path vertex) --------------------------
template <int K> struct Du {
  float v;
  float d[K];
};
template <int K> __device__ __forceinline__ Du<K> du_const(float c) { Du<K> r; r.v = c; for (int i = 0; i < K; ++i) r.d[i] = 0.f; return r; }
template <int K> __device__ __forceinline__ Du<K> du_var(float c, int k) { Du<K> r = du_const<K>(c); r.d[k] = 1.f; return r; }
template <int K> __device__ __forceinline__ Du<K> operator+(Du<K> a, Du<K> b) { Du<K> r; r.v = a.v + b.v; for (int i = 0; i < K; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
template <int K> __device__ __forceinline__ Du<K> operator-(Du<K> a, Du<K> b) { Du<K> r; r.v = a.v - b.v; for (int i = 0; i < K; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
template <int K> __device__ __forceinline__ Du<K> operator-(Du<K> a) { Du<K> r; r.v = -a.v; for (int i = 0; i < K; ++i) r.d[i] = -a.d[i]; return r; }
template <int K> __device__ __forceinline__ Du<K> operator*(Du<K> a, Du<K> b) { Du<K> r; r.v = a.v * b.v; for (int i = 0; i < K; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
template <int K> __device__ __forceinline__ Du<K> operator*(Du<K> a, float b) { Du<K> r; r.v = a.v * b; for (int i = 0; i < K; ++i) r.d[i] = a.d[i] * b; return r; }
template <int K> __device__ __forceinline__ Du<K> operator*(float b, Du<K> a) { return a * b; }
template <int K> __device__ __forceinline__ Du<K> operator+(Du<K> a, float b) { a.v += b; return a; }
template <int K> __device__ __forceinline__ Du<K> operator+(float b, Du<K> a) { a.v += b; return a; }
template <int K> __device__ __forceinline__ Du<K> operator-(Du<K> a, float b) { a.v -= b; return a; }
template <int K> __device__ __forceinline__ Du<K> operator-(float b, Du<K> a) { return (-a) + b; }
template <int K> __device__ __forceinline__ Du<K> operator/(Du<K> a, Du<K> b) {
  Du<K> r; const float inv = 1.0f / b.v; r.v = a.v * inv;
  for (int i = 0; i < K; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) * inv;
  return r;
}
template <int K> __device__ __forceinline__ Du<K> operator/(float a, Du<K> b) { return du_const<K>(a) / b; }
template <int K> __device__ __forceinline__ Du<K> sqrt_t(Du<K> a) {
  Du<K> r; r.v = sqrtf(a.v); const float k = a.v > 0.f ? 0.5f / r.v : 0.f;
  for (int i = 0; i < K; ++i) r.d[i] = a.d[i] * k;
  return r;
}
template <int K> __device__ __forceinline__ void sincos_t(Du<K> a, Du<K>& s, Du<K>& c) {
  float sv, cv; sincosf(a.v, &sv, &cv);
  s.v = sv; c.v = cv;
  for (int i = 0; i < K; ++i) { s.d[i] = a.d[i] * cv; c.d[i] = -a.d[i] * sv; }
}
template <int K> __device__ __forceinline__ float val(Du<K> a) { return a.v; }
template <int K> __device__ __forceinline__ Du<K> clamp0(Du<K> a) { return a.v < 0.f ? du_const<K>(0.f) : a; }
__device__ __forceinline__ float sqrt_t(float a) { return sqrtf(a); }
__device__ __forceinline__ void sincos_t(float a, float& s, float& c) { sincosf(a, &s, &c); }
__device__ __forceinline__ float val(float a) { return a; }
__device__ __forceinline__ float clamp0(float a) { return a < 0.f ? 0.f : a; }

template <class T> struct V3 { T x, y, z; };
template <class T> __device__ __forceinline__ T dotf(V3<T> a, float3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> __device__ __forceinline__ T dott(V3<T> a, V3<T> b) { return a.x * b.x + a.y * b.y + a.z * b.z; }

// ---- a4: closest hit over the BVH8 ----------------------------------------------------------------------
struct HitRec {
  float t;
  uint32_t li;  // triangle in leaf order; 0xFFFFFFFF = miss
};

// Moeller-Trumbore, no culling, t > 0, tie: smaller t then smaller original id (Q8).
__device__ __forceinline__ void test_tri(const float4* __restrict__ tris, uint32_t li, float3 o, float3 d, HitRec& best,
                                         uint32_t& best_id) {
  const float4 q0 = __ldg(&tris[3 * li]), q1 = __ldg(&tris[3 * li + 1]), q2 = __ldg(&tris[3 * li + 2]);
  const float3 e1 = xyz(q1), e2 = xyz(q2);
  const float3 pv = cross3(d, e2);
  const float det = dot3(e1, pv);
  if (det == 0.f) return;
  const float inv = 1.0f / det;
  const float3 tv = o - xyz(q0);
  const float u = dot3(tv, pv) * inv;
  if (u < 0.f || u > 1.f) return;
  const float3 qv = cross3(tv, e1);
  const float v = dot3(d, qv) * inv;
  if (v < 0.f || u + v > 1.f) return;
  const float t = dot3(e2, qv) * inv;
  if (!(t > 0.f)) return;
  const uint32_t id = __float_as_uint(q0.w);
  if (t < best.t || (t == best.t && id < best_id)) { best.t = t; best.li = li; best_id = id; }
}

// One lane = one ray.  snodes: the first sc.smem_nodes nodes staged in shared memory (may be null if 0).
template <bool STATS = false>
__device__ __forceinline__ HitRec closest_hit(const DevScene& sc, const float4* snodes, float3 o, float3 d,
                                              uint32_t* n_nodes = nullptr, uint32_t* n_tris = nullptr) {
  HitRec best{FLT_MAX, 0xFFFFFFFFu};
  uint32_t best_id = 0xFFFFFFFFu;
  // box tests use a direction with no zero component (finite reciprocals); triangle tests use d itself
  const float dxs = fabsf(d.x) < 1e-20f ? copysignf(1e-20f, d.x) : d.x;
  const float dys = fabsf(d.y) < 1e-20f ? copysignf(1e-20f, d.y) : d.y;
  const float dzs = fabsf(d.z) < 1e-20f ? copysignf(1e-20f, d.z) : d.z;
  const float ix = 1.0f / dxs, iy = 1.0f / dys, iz = 1.0f / dzs;
  const float ox = o.x * ix, oy = o.y * iy, oz = o.z * iz;
  uint32_t st_n[kStackDepth];
  float st_t[kStackDepth];
  int sp = 0;
  uint32_t cur = 0;  // root
  for (;;) {
    if (!(cur & kLeafBit)) {
      const float4* np = cur < sc.smem_nodes ? snodes + 16 * cur : sc.nodes + 16 * (size_t)cur;
      if (STATS) ++*n_nodes;
      float tn[8];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const float4 lx = np[0 + h], ly = np[2 + h], lz = np[4 + h];
        const float4 hx = np[6 + h], hy = np[8 + h], hz = np[10 + h];
        const float lxa[4] = {lx.x, lx.y, lx.z, lx.w}, lya[4] = {ly.x, ly.y, ly.z, ly.w}, lza[4] = {lz.x, lz.y, lz.z, lz.w};
        const float hxa[4] = {hx.x, hx.y, hx.z, hx.w}, hya[4] = {hy.x, hy.y, hy.z, hy.w}, hza[4] = {hz.x, hz.y, hz.z, hz.w};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const float ax = fmaf(lxa[c], ix, -ox), bx = fmaf(hxa[c], ix, -ox);
          const float ay = fmaf(lya[c], iy, -oy), by = fmaf(hya[c], iy, -oy);
          const float az = fmaf(lza[c], iz, -oz), bz = fmaf(hza[c], iz, -oz);
          const float tmin = fmaxf(fmaxf(fminf(ax, bx), fminf(ay, by)), fmaxf(fminf(az, bz), 0.f));
          const float tmax = fminf(fminf(fmaxf(ax, bx), fmaxf(ay, by)), fminf(fmaxf(az, bz), best.t));
          tn[4 * h + c] = tmin <= tmax ? tmin : FLT_MAX;  // empty slots are far-away point boxes: never hit
        }
      }
      const uint4 c0 = *reinterpret_cast<const uint4*>(np + 12), c1 = *reinterpret_cast<const uint4*>(np + 13);
      const uint32_t ch[8] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
      // descend into the nearest hit child, push the others
      float near_t = FLT_MAX;
      uint32_t near_c = kEmptyChild;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (tn[i] != FLT_MAX) {
          uint32_t pc = ch[i];
          float pt = tn[i];
          if (pt < near_t) {
            const uint32_t oc = near_c; const float ot = near_t;
            near_c = pc; near_t = pt; pc = oc; pt = ot;
          }
          if (pc != kEmptyChild && sp < kStackDepth) { st_n[sp] = pc; st_t[sp] = pt; ++sp; }
        }
      }
      if (near_c != kEmptyChild) { cur = near_c; continue; }
    } else {
      const uint32_t first = cur & 0x07FFFFFFu, cnt = ((cur >> 27) & 0xFu) + 1u;
      for (uint32_t k = 0; k < cnt; ++k) test_tri(sc.tris, first + k, o, d, best, best_id);
      if (STATS) *n_tris += cnt;
    }
    // pop the next entry that can still contain a closer (or tying) hit
    bool found = false;
    while (sp > 0) {
      --sp;
      if (st_t[sp] <= best.t) { cur = st_n[sp]; found = true; break; }
    }
    if (!found) break;
  }
  return best;
}

// ---- a3 / a5: materials ---------------------------------------------------------------------------------
struct Frame {
  float3 t, bf, nf;  // tangent, bitangent and normal facing the incoming ray (Q6)
};

__device__ __forceinline__ void tri_frame(float3 e1, float3 e2, float3 din, Frame& fr, float& dn) {
  const float3 tg = normalize3(e1);
  const float3 n = normalize3(cross3(e1, e2));
  const float3 bt = cross3(n, tg);
  dn = dot3(din, n);
  const float side = dn < 0.f ? 1.f : -1.f;
  fr.t = tg; fr.bf = bt * side; fr.nf = n * side;
}

template <class T> __device__ __forceinline__ V3<T> from_frame(const Frame& fr, T wx, T wy, T wz) {
  V3<T> r;
  r.x = wx * fr.t.x + wy * fr.bf.x + wz * fr.nf.x;
  r.y = wx * fr.t.y + wy * fr.bf.y + wz * fr.nf.y;
  r.z = wx * fr.t.z + wy * fr.bf.z + wz * fr.nf.z;
  return r;
}

// Lambert: cosine-weighted direction from (u1, u2); weight = albedo (constant).
template <class T> __device__ __forceinline__ V3<T> lambert_dir(const Frame& fr, T u1, T u2) {
  const T r = sqrt_t(u1);
  T s, c;
  sincos_t(u2 * kTwoPi, s, c);
  return from_frame<T>(fr, r * c, r * s, sqrt_t(1.0f - u1));
}

// Exact unpolarised Fresnel for a smooth dielectric, eta = n_t / n_i.
__device__ __forceinline__ float fresnel_dielectric(float cos_i, float eta) {
  const float sin2_t = (1.0f - cos_i * cos_i) / (eta * eta);
  if (sin2_t >= 1.0f) return 1.0f;
  const float cos_t = sqrtf(1.0f - sin2_t);
  const float r_par = (eta * cos_i - cos_t) / (eta * cos_i + cos_t);
  const float r_perp = (cos_i - eta * cos_t) / (cos_i + eta * cos_t);
  return 0.5f * (r_par * r_par + r_perp * r_perp);
}

template <class T> __device__ __forceinline__ V3<T> dielectric_dir(const Frame& fr, float eta, bool reflect, V3<T> d) {
  const T cos_i = -dotf(d, fr.nf);
  V3<T> r;
  if (reflect) {
    const T k = cos_i * 2.0f;
    r.x = d.x + k * fr.nf.x; r.y = d.y + k * fr.nf.y; r.z = d.z + k * fr.nf.z;
  } else {
    const float ie = 1.0f / eta;
    const T ct = sqrt_t(1.0f - (1.0f - cos_i * cos_i) * (ie * ie));
    const T k = cos_i * ie - ct;
    r.x = d.x * ie + k * fr.nf.x; r.y = d.y * ie + k * fr.nf.y; r.z = d.z * ie + k * fr.nf.z;
  }
  return r;
}

// GGX conductor: visible-normal sampling (spherical-cap form).  Returns false if w_i is below the horizon.
// c5 = (1 - w_o.h)^5 (Schlick), G1 = Smith masking of w_i; weight_c = (F0_c + (1 - F0_c) c5) G1.
template <class T> __device__ __forceinline__ bool ggx_dir(const Frame& fr, float al, V3<T> d, T u1, T u2, V3<T>& out, T& c5, T& G1) {
  V3<T> wo;
  wo.x = -dotf(d, fr.t); wo.y = -dotf(d, fr.bf); wo.z = -dotf(d, fr.nf);
  V3<T> ws;
  ws.x = wo.x * al; ws.y = wo.y * al; ws.z = wo.z;
  const T wsn = 1.0f / sqrt_t(dott(ws, ws));
  ws.x = ws.x * wsn; ws.y = ws.y * wsn; ws.z = ws.z * wsn;
  T s, c;
  sincos_t(u2 * kTwoPi, s, c);
  const T z = (1.0f - u1) * (1.0f + ws.z) - ws.z;
  const T st = sqrt_t(clamp0(1.0f - z * z));
  V3<T> hm;
  hm.x = (st * c + ws.x) * al; hm.y = (st * s + ws.y) * al; hm.z = z + ws.z;
  const T hn = 1.0f / sqrt_t(dott(hm, hm));
  hm.x = hm.x * hn; hm.y = hm.y * hn; hm.z = hm.z * hn;
  const T woh = dott(wo, hm);
  V3<T> wi;
  const T k2 = woh * 2.0f;
  wi.x = hm.x * k2 - wo.x; wi.y = hm.y * k2 - wo.y; wi.z = hm.z * k2 - wo.z;
  if (!(val(wi.z) > 0.f)) return false;
  const T c1 = 1.0f - woh;
  const T c2 = c1 * c1;
  c5 = c2 * c2 * c1;
  G1 = (wi.z * 2.0f) / (wi.z + sqrt_t((wi.x * wi.x + wi.y * wi.y) * (al * al) + wi.z * wi.z));
  out = from_frame<T>(fr, wi.x, wi.y, wi.z);
  return true;
}

template <class T> __device__ __forceinline__ V3<T> camera_dir(const DevScene& sc, T x0, T x1) {
  const T sx = (x0 * 2.0f - 1.0f) * sc.tan_half_aspect;
  const T sy = (x1 * 2.0f - 1.0f) * sc.tan_half;
  V3<T> v;
  v.x = sx * sc.cam_r[0] - sy * sc.cam_v[0] + sc.cam_w[0];
  v.y = sx * sc.cam_r[1] - sy * sc.cam_v[1] + sc.cam_w[1];
  v.z = sx * sc.cam_r[2] - sy * sc.cam_v[2] + sc.cam_w[2];
  const T inv = 1.0f / sqrt_t(dott(v, v));
  v.x = v.x * inv; v.y = v.y * inv; v.z = v.z * inv;
  return v;
}

__device__ __forceinline__ uint32_t fnv(uint32_t h, uint32_t v) { return (h ^ v) * 16777619u; }

__device__ __forceinline__ uint32_t pixel_of(float x0, float x1, uint32_t W, uint32_t H) {
  const uint32_t px = min((uint32_t)floorf(x0 * (float)W), W - 1u);
  const uint32_t py = min((uint32_t)floorf(x1 * (float)H), H - 1u);
  return py * W + px;
}

struct EvalOut {
  float f[3];
  float p;
  uint32_t pix, nrays, sig;
  bool nonfinite;
};

// Access to the d PSS coordinates of one state: SoA planes (float4[plane * stride + idx]) or a row-major row.
struct XView {
  const float4* planes;  // null -> row-major
  const float* row;
  size_t stride;
  size_t idx;
  __device__ __forceinline__ float2 pair(uint32_t k) const {  // coordinates (2k, 2k+1)
    if (planes) {
      const float4 q = planes[(size_t)(k >> 1) * stride + idx];
      return (k & 1u) ? make_float2(q.z, q.w) : make_float2(q.x, q.y);
    }
    return make_float2(row[2 * k], row[2 * k + 1]);
  }
};

// Writes the score pair of vertex k (coordinates 2k, 2k+1).
struct GView {
  float4* planes;
  float* row;
  size_t stride;
  size_t idx;
  __device__ __forceinline__ void pair(uint32_t k, float a, float b) const {
    if (planes) {
      float2* q = reinterpret_cast<float2*>(&planes[(size_t)(k >> 1) * stride + idx]);
      q[k & 1u] = make_float2(a, b);
    } else if (row) {
      row[2 * k] = a; row[2 * k + 1] = b;
    }
  }
};

__device__ __forceinline__ float min_image(float v) { return v - floorf(v + 0.5f); }

// 2-D analytic target (wrapped-Gaussian mixture), see dr.h dr_analytic2d_desc.
__device__ __forceinline__ void wrapped_gauss(float delta, float s, float& w, float& dw) {
  w = 0.f; dw = 0.f;
  const float inv = 1.0f / s, norm = 0.3989422804014327f * inv;
#pragma unroll
  for (int j = -2; j <= 2; ++j) {
    const float z = (delta + (float)j) * inv;
    const float e = norm * expf(-0.5f * z * z);
    w += e;
    dw += -z * inv * e;
  }
}

template <bool GRAD>
__device__ void eval_analytic(const DevScene& sc, const XView& xv, EvalOut& out, const GView& gv) {
  const float2 x = xv.pair(0);
  float p = 0.f, gx = 0.f, gy = 0.f;
  for (int k = 0; k < sc.n_mix; ++k) {
    float wx, dwx, wy, dwy;
    wrapped_gauss(min_image(x.x - sc.mix_mx[k]), sc.mix_s[k], wx, dwx);
    wrapped_gauss(min_image(x.y - sc.mix_my[k]), sc.mix_s[k], wy, dwy);
    p += sc.mix_w[k] * wx * wy;
    gx += sc.mix_w[k] * dwx * wy;
    gy += sc.mix_w[k] * wx * dwy;
  }
  out.f[0] = out.f[1] = out.f[2] = out.p = p;
  out.pix = pixel_of(x.x, x.y, sc.W, sc.H);
  out.nrays = 0; out.sig = 0;
  float g0 = gx / (p + kEps), g1 = gy / (p + kEps);
  out.nonfinite = !(isfinite(p)) || (GRAD && !(isfinite(g0) && isfinite(g1)));
  if (out.nonfinite) { out.f[0] = out.f[1] = out.f[2] = out.p = 0.f; g0 = g1 = 0.f; }
  if (GRAD) gv.pair(0, g0, g1);
}

// Path evaluation.  GRAD: also the score, written through gv for all L vertex slots.
template <bool GRAD, bool STATS = false>
__device__ void eval_path(const DevScene& sc, const float4* snodes, const XView& xv, EvalOut& out, const GView& gv,
                          uint32_t* n_nodes = nullptr, uint32_t* n_tris = nullptr) {
  const uint32_t L = sc.L;
  // per-vertex record for the reverse pass (local memory; only touched when GRAD)
  float3 rec_d[GRAD ? kMaxPathLen : 1];
  uint32_t rec_li[GRAD ? kMaxPathLen : 1];
  uint32_t refract_mask = 0, ggx_mask = 0;
  uint32_t nvert = 0;  // vertices at which a direction was sampled (1..nvert)

  const float2 x01 = xv.pair(0);
  out.pix = pixel_of(x01.x, x01.y, sc.W, sc.H);
  out.nrays = 0;
  uint32_t sig = 2166136261u;
  const V3<float> d0 = camera_dir<float>(sc, x01.x, x01.y);
  float3 d = make_float3(d0.x, d0.y, d0.z);
  float3 o = make_float3(sc.cam_pos[0], sc.cam_pos[1], sc.cam_pos[2]);
  float T0 = 1.f, T1 = 1.f, T2 = 1.f;
  float f0 = 0.f, f1 = 0.f, f2 = 0.f;

  for (uint32_t k = 1; k <= L; ++k) {
    const HitRec h = closest_hit<STATS>(sc, snodes, o, d, n_nodes, n_tris);
    ++out.nrays;
    if (h.li == 0xFFFFFFFFu) {
      sig = fnv(sig, 0u);
      f0 = T0 * sc.env[0]; f1 = T1 * sc.env[1]; f2 = T2 * sc.env[2];
      break;
    }
    const float4 q0 = __ldg(&sc.tris[3 * h.li]), q1 = __ldg(&sc.tris[3 * h.li + 1]), q2 = __ldg(&sc.tris[3 * h.li + 2]);
    sig = fnv(sig, __float_as_uint(q0.w) + 1u);
    const uint32_t mi = __float_as_uint(q1.w);
    const float4 m0 = __ldg(&sc.mats[3 * mi]), m1 = __ldg(&sc.mats[3 * mi + 1]);
    const uint32_t kind = __float_as_uint(m0.x);
    Frame fr;
    float dn;
    tri_frame(xyz(q1), xyz(q2), d, fr, dn);
    if (kind == 3u) {  // emitter: front face emits, path stops
      if (dn < 0.f) {
        sig = fnv(sig, 4u);
        const float4 m2 = __ldg(&sc.mats[3 * mi + 2]);
        f0 = T0 * m1.z; f1 = T1 * m1.w; f2 = T2 * m2.x;
      } else {
        sig = fnv(sig, 5u);
      }
      break;
    }
    if (k == L) break;
    const float3 hit = o + d * h.t;
    const float2 u = xv.pair(k);
    if (GRAD) { rec_d[k] = d; rec_li[k] = h.li; }
    nvert = k;
    V3<float> din{d.x, d.y, d.z}, dnew;
    float off = 1.f;
    if (kind == 0u) {
      sig = fnv(sig, 0u);
      dnew = lambert_dir<float>(fr, u.x, u.y);
      T0 *= m0.y; T1 *= m0.z; T2 *= m0.w;
    } else if (kind == 1u) {
      const float eta = dn < 0.f ? m1.x : 1.0f / m1.x;
      const float F = fresnel_dielectric(-dot3(d, fr.nf), eta);
      const bool reflect = u.x < F;
      sig = fnv(sig, reflect ? 1u : 2u);
      if (!reflect) { off = -1.f; refract_mask |= 1u << k; }
      dnew = dielectric_dir<float>(fr, eta, reflect, din);
    } else {
      sig = fnv(sig, 3u);
      ggx_mask |= 1u << k;
      float c5, G1;
      if (!ggx_dir<float>(fr, m1.y, din, u.x, u.y, dnew, c5, G1)) {
        T0 = T1 = T2 = 0.f;
      } else {
        T0 *= (m0.y + (1.0f - m0.y) * c5) * G1;
        T1 *= (m0.z + (1.0f - m0.z) * c5) * G1;
        T2 *= (m0.w + (1.0f - m0.w) * c5) * G1;
      }
    }
    if (T0 == 0.f && T1 == 0.f && T2 == 0.f) break;
    o = hit + fr.nf * (sc.eps_ray * off);
    d = make_float3(dnew.x, dnew.y, dnew.z);
  }
  float p = f0 * 0.2126f + f1 * 0.7152f + f2 * 0.0722f;
  out.sig = sig;
  out.nonfinite = !(isfinite(f0) && isfinite(f1) && isfinite(f2) && isfinite(p));
  if (out.nonfinite) { f0 = f1 = f2 = p = 0.f; }
  out.f[0] = f0; out.f[1] = f1; out.f[2] = f2; out.p = p;
  if (!GRAD) return;

  // ---- a6: score by reverse accumulation ------------------------------------------------------------
  // Only GGX weights depend on x: no GGX vertex or p == 0  =>  g == 0 exactly.
  if (ggx_mask == 0u || !(p > 0.f)) {
    for (uint32_t k = 0; k < L; ++k) gv.pair(k, 0.f, 0.f);
    return;
  }
  const float inv_phat = 1.0f / (p + kEps);
  const float A0 = 0.2126f * f0, A1 = 0.7152f * f1, A2 = 0.0722f * f2;  // d p / d ln(w_c) per channel
  float db0 = 0.f, db1 = 0.f, db2 = 0.f;  // adjoint of the outgoing direction of the current vertex
  bool bad = false;
  for (uint32_t k = L - 1; k >= 1; --k) {
    float ga = 0.f, gb = 0.f;
    if (k <= nvert) {
      const uint32_t li = rec_li[k];
      const float3 din = rec_d[k];
      const float4 q1 = __ldg(&sc.tris[3 * li + 1]), q2 = __ldg(&sc.tris[3 * li + 2]);
      const uint32_t mi = __float_as_uint(q1.w);
      const float4 m0 = __ldg(&sc.mats[3 * mi]), m1 = __ldg(&sc.mats[3 * mi + 1]);
      const uint32_t kind = __float_as_uint(m0.x);
      Frame fr;
      float dn;
      tri_frame(xyz(q1), xyz(q2), din, fr, dn);
      const float2 u = xv.pair(k);
      const bool live = db0 != 0.f || db1 != 0.f || db2 != 0.f;
      if (kind == 0u) {
        if (live) {
          const V3<Du<2>> w = lambert_dir<Du<2>>(fr, du_var<2>(u.x, 0), du_var<2>(u.y, 1));
          ga = db0 * w.x.d[0] + db1 * w.y.d[0] + db2 * w.z.d[0];
          gb = db0 * w.x.d[1] + db1 * w.y.d[1] + db2 * w.z.d[1];
        }
        db0 = db1 = db2 = 0.f;  // a diffuse vertex forgets the incoming direction
      } else if (kind == 1u) {
        if (live) {
          const float eta = dn < 0.f ? m1.x : 1.0f / m1.x;
          V3<Du<3>> di{du_var<3>(din.x, 0), du_var<3>(din.y, 1), du_var<3>(din.z, 2)};
          const V3<Du<3>> w = dielectric_dir<Du<3>>(fr, eta, !((refract_mask >> k) & 1u), di);
          const float n0 = db0 * w.x.d[0] + db1 * w.y.d[0] + db2 * w.z.d[0];
          const float n1 = db0 * w.x.d[1] + db1 * w.y.d[1] + db2 * w.z.d[1];
          const float n2 = db0 * w.x.d[2] + db1 * w.y.d[2] + db2 * w.z.d[2];
          db0 = n0; db1 = n1; db2 = n2;
        }
      } else if (kind == 2u) {
        V3<Du<5>> di{du_var<5>(din.x, 2), du_var<5>(din.y, 3), du_var<5>(din.z, 4)};
        V3<Du<5>> w;
        Du<5> c5, G1;
        if (ggx_dir<Du<5>>(fr, m1.y, di, du_var<5>(u.x, 0), du_var<5>(u.y, 1), w, c5, G1)) {
          // S = sum_c (A_c / w_c) w_c(x) with w_c = (F0_c + (1 - F0_c) c5) G1
          const float w0 = (m0.y + (1.0f - m0.y) * c5.v) * G1.v, w1 = (m0.z + (1.0f - m0.z) * c5.v) * G1.v,
                      w2 = (m0.w + (1.0f - m0.w) * c5.v) * G1.v;
          const float B0 = w0 > 0.f ? A0 / w0 : 0.f, B1 = w1 > 0.f ? A1 / w1 : 0.f, B2 = w2 > 0.f ? A2 / w2 : 0.f;
          const float a0 = B0 * m0.y + B1 * m0.z + B2 * m0.w;
          const float a1 = B0 * (1.0f - m0.y) + B1 * (1.0f - m0.z) + B2 * (1.0f - m0.w);
          const Du<5> S = G1 * (c5 * a1 + a0);
          float n[5];
#pragma unroll
          for (int j = 0; j < 5; ++j) n[j] = db0 * w.x.d[j] + db1 * w.y.d[j] + db2 * w.z.d[j] + S.d[j];
          ga = n[0]; gb = n[1];
          db0 = n[2]; db1 = n[3]; db2 = n[4];
        }
      }
    }
    ga *= inv_phat; gb *= inv_phat;
    bad = bad || !(isfinite(ga) && isfinite(gb));
    gv.pair(k, ga, gb);
  }
  {
    float ga = 0.f, gb = 0.f;
    if (db0 != 0.f || db1 != 0.f || db2 != 0.f) {
      const V3<Du<2>> w = camera_dir<Du<2>>(sc, du_var<2>(x01.x, 0), du_var<2>(x01.y, 1));
      ga = (db0 * w.x.d[0] + db1 * w.y.d[0] + db2 * w.z.d[0]) * inv_phat;
      gb = (db0 * w.x.d[1] + db1 * w.y.d[1] + db2 * w.z.d[1]) * inv_phat;
    }
    bad = bad || !(isfinite(ga) && isfinite(gb));
    gv.pair(0, ga, gb);
  }
  if (bad) {  // Q18: a non-finite score makes the state a zero-contribution state
    out.nonfinite = true;
    out.f[0] = out.f[1] = out.f[2] = out.p = 0.f;
    for (uint32_t k = 0; k < L; ++k) gv.pair(k, 0.f, 0.f);
  }
}

}  // namespace dr
