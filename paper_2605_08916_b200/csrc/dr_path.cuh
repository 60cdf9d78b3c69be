// Arithmetic note: the library is compiled with -fmad=false (build.py), and the value formulas below are written in the
// operation order of DESIGN.md Q4-Q8, so that a path's hit points, directions and weights round exactly as a plain fp32
// evaluation of those formulas does; only sincosf / logf (a few ulps) can differ.  Near-threshold decisions (which facet
// an edge-grazing ray hits) then fall the same way on both sides of a parity check (Q15).
// Target evaluation on the device, per-vertex pieces: x -> (f, p, pixel, score)  (rows a3, a5, a6).
//   a3 camera ray and direction sampling at a vertex, a5 throughput / emission, a6 the local Jacobians of the
//   reverse pass (forward-mode numbers with a handful of tangents).  One vertex as a whole is vertex_fn (dr_nee.cuh); the
//   wavefront kernels that call these are in dr_eval.cuh / dr_wave.cuh / dr_grad.cuh; the closest-hit query (a4) is dr_traverse.cuh.
// The path map is DESIGN.md Q4-Q9 (the paper does not describe its path sampling routines).
#pragma once
#include <cfloat>
#include <cstdint>
#include <cuda_runtime.h>

#include "dr_types.h"

namespace dr {

constexpr float kEps = 1e-8f;
constexpr float kTwoPi = 6.283185307179586f;

struct DevScene {
  const uint4* nodes;   // NodeC as 5 uint4
  const float4* tris;   // TriPacked as 3 float4
  const float4* mats;   // MatPacked as 3 float4
  uint32_t n_nodes, stack_cap, n_tris, n_mats;
  const float4* lights; // next-event estimation (dr_nee.cuh Light): 5 float4 per emitter triangle
  uint32_t n_lights, nee;
  float light_total;
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
template <int K> __device__ __forceinline__ Du<K> operator/(Du<K> a, float b) { Du<K> r; r.v = a.v / b; for (int i = 0; i < K; ++i) r.d[i] = a.d[i] / b; return r; }
template <int K> __device__ __forceinline__ Du<K> sqrt_t(Du<K> a) {
  Du<K> r; r.v = sqrtf(a.v); const float k = a.v > 0.f ? 0.5f / r.v : 0.f;
  for (int i = 0; i < K; ++i) r.d[i] = a.d[i] * k;
  return r;
}
#ifndef DR_SINCOS_F64
#define DR_SINCOS_F64 0
#endif
// sin and cos of an angle in [0, 2 pi).  DR_SINCOS_F64: evaluated in double and rounded once, i.e. the correctly rounded
// fp32 values (what a good host libm returns); otherwise sincosf (2 ulp).
__device__ __forceinline__ void sincos_f(float a, float* s, float* c) {
#if DR_SINCOS_F64
  double sd, cd;
  sincos((double)a, &sd, &cd);
  *s = (float)sd; *c = (float)cd;
#else
  sincosf(a, s, c);
#endif
}
template <int K> __device__ __forceinline__ void sincos_t(Du<K> a, Du<K>& s, Du<K>& c) {
  float sv, cv; sincos_f(a.v, &sv, &cv);
  s.v = sv; c.v = cv;
  for (int i = 0; i < K; ++i) { s.d[i] = a.d[i] * cv; c.d[i] = -a.d[i] * sv; }
}
template <int K> __device__ __forceinline__ float val(Du<K> a) { return a.v; }
template <int K> __device__ __forceinline__ Du<K> clamp0(Du<K> a) { return a.v < 0.f ? du_const<K>(0.f) : a; }
__device__ __forceinline__ float sqrt_t(float a) { return sqrtf(a); }
__device__ __forceinline__ void sincos_t(float a, float& s, float& c) { sincos_f(a, &s, &c); }
__device__ __forceinline__ float val(float a) { return a; }
__device__ __forceinline__ float clamp0(float a) { return a < 0.f ? 0.f : a; }

template <class T> struct V3 { T x, y, z; };
template <class T> __device__ __forceinline__ T dotf(V3<T> a, float3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> __device__ __forceinline__ T dott(V3<T> a, V3<T> b) { return a.x * b.x + a.y * b.y + a.z * b.z; }

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
    const T ct = sqrt_t(1.0f - (1.0f - cos_i * cos_i) / (eta * eta));
    const T k = cos_i / eta - ct;
    r.x = d.x * ie + k * fr.nf.x; r.y = d.y * ie + k * fr.nf.y; r.z = d.z * ie + k * fr.nf.z;
  }
  return r;
}

// GGX conductor: visible-normal sampling (spherical-cap form).  Returns false if w_i is below the horizon.
// c5 = (1 - w_o.h)^5 (Schlick), G1 = Smith masking of w_i; weight_c = (F0_c + (1 - F0_c) c5) G1.
template <class T> __device__ __forceinline__ bool ggx_dir(const Frame& fr, float al, V3<T> d, T u1, T u2, V3<T>& out, T& c5, T& G1,
                                                           V3<T>* hm_out = nullptr) {
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
  if (hm_out) *hm_out = hm;
  const T woh = dott(wo, hm);
  V3<T> wi;
  const T k2 = woh * 2.0f;
  wi.x = hm.x * k2 - wo.x; wi.y = hm.y * k2 - wo.y; wi.z = hm.z * k2 - wo.z;
  if (!(val(wi.z) > 0.f)) return false;
  const T c1 = 1.0f - woh;
  c5 = c1 * c1 * c1 * c1 * c1;
  G1 = (wi.z * 2.0f) / (wi.z + sqrt_t((wi.x * wi.x + wi.y * wi.y) * (al * al) + wi.z * wi.z));
  out = from_frame<T>(fr, wi.x, wi.y, wi.z);
  return true;
}

template <class T> __device__ __forceinline__ V3<T> camera_dir(const DevScene& sc, T x0, T x1) {
  const T sx = (x0 * 2.0f - 1.0f) * sc.tan_half_aspect;
  const T sy = (x1 * 2.0f - 1.0f) * sc.tan_half;
  V3<T> v;
  v.x = (sc.cam_w[0] + sx * sc.cam_r[0]) - sy * sc.cam_v[0];
  v.y = (sc.cam_w[1] + sx * sc.cam_r[1]) - sy * sc.cam_v[1];
  v.z = (sc.cam_w[2] + sx * sc.cam_r[2]) - sy * sc.cam_v[2];
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

// p, its gradient over (p + eps), and the pixel of one state of the analytic target.
__device__ __forceinline__ void eval_analytic(const DevScene& sc, float x0, float x1, float& p_out, float& g0, float& g1) {
  float p = 0.f, gx = 0.f, gy = 0.f;
  for (int k = 0; k < sc.n_mix; ++k) {
    float wx, dwx, wy, dwy;
    wrapped_gauss(min_image(x0 - sc.mix_mx[k]), sc.mix_s[k], wx, dwx);
    wrapped_gauss(min_image(x1 - sc.mix_my[k]), sc.mix_s[k], wy, dwy);
    p += sc.mix_w[k] * wx * wy;
    gx += sc.mix_w[k] * dwx * wy;
    gy += sc.mix_w[k] * wx * dwy;
  }
  p_out = p;
  g0 = gx / (p + kEps);
  g1 = gy / (p + kEps);
}

}  // namespace dr
