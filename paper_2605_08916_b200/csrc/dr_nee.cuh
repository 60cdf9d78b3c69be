// One path vertex as a function (rows a3 / a5 / a6 with next-event estimation, Q21):
//   (ray that arrived: o, d; the vertex' four coordinates u1, u2, v1, v2)  ->
//   (next ray o2, d2; density pb of its direction; throughput factor W; emitter connection C per unit throughput)
// written once for T = float (the shading of the wavefront kernels) and T = Du<K> (the local Jacobians of the score's
// reverse sweep, dr_grad.cuh).  The triangle, the side it was hit from, the dielectric lobe, the emitter triangle and
// the visibility are discrete: decided on the values by the float instantiation, given to the Du one.
// Value arithmetic in the operation order of DESIGN.md Q4-Q8 / Q21 (the library is built with -fmad=false).
#pragma once
#include "dr_path.cuh"

namespace dr {

constexpr float kInvPi = 0.31830988618379067f;

template <class T> __device__ __forceinline__ V3<T> vsubf(float3 a, V3<T> b) { V3<T> r; r.x = a.x - b.x; r.y = a.y - b.y; r.z = a.z - b.z; return r; }
template <class T> __device__ __forceinline__ V3<T> vsub(V3<T> a, V3<T> b) { V3<T> r; r.x = a.x - b.x; r.y = a.y - b.y; r.z = a.z - b.z; return r; }
template <class T> __device__ __forceinline__ V3<T> vadd(V3<T> a, V3<T> b) { V3<T> r; r.x = a.x + b.x; r.y = a.y + b.y; r.z = a.z + b.z; return r; }
template <class T> __device__ __forceinline__ V3<T> vscale(V3<T> a, T s) { V3<T> r; r.x = a.x * s; r.y = a.y * s; r.z = a.z * s; return r; }
template <class T> __device__ __forceinline__ V3<T> vnormalize(V3<T> a) { const T inv = 1.0f / sqrt_t(dott(a, a)); return vscale(a, inv); }
template <class T> __device__ __forceinline__ T lift_t(float c);
template <> __device__ __forceinline__ float lift_t<float>(float c) { return c; }
template <class T> __device__ __forceinline__ T lift_t(float c) { T r; r.v = c; for (int i = 0; i < (int)(sizeof(r.d) / sizeof(float)); ++i) r.d[i] = 0.f; return r; }

// Smith G1 of the separable GGX masking, local frame (z = normal).
template <class T> __device__ __forceinline__ T ggx_g1(V3<T> w, float al) {
  return (w.z * 2.0f) / (w.z + sqrt_t((w.x * w.x + w.y * w.y) * (al * al) + w.z * w.z));
}
// GGX normal distribution D(h), local frame.
template <class T> __device__ __forceinline__ T ggx_d(V3<T> h, float al) {
  const T q = h.z * h.z * (al * al - 1.0f) + 1.0f;
  return (al * al * kInvPi) / (q * q);
}

// Emitter list (DevScene::lights): five float4 per emitter triangle, in triangle-index order:
//   (v0, running area sum up to and including it) (e1, area) (e2, bits(triangle id)) (unit normal, running sum before it) (Le, 0)
struct Light {
  float3 v0, e1, e2, n, le;
  float cdf, before, area;
  uint32_t id;
};
__device__ __forceinline__ Light load_light(const DevScene& sc, uint32_t j) {
  const float4* p = sc.lights + 5 * (size_t)j;
  const float4 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2), d = __ldg(p + 3), e = __ldg(p + 4);
  Light L;
  L.v0 = xyz(a); L.cdf = a.w; L.e1 = xyz(b); L.area = b.w; L.e2 = xyz(c); L.id = __float_as_uint(c.w);
  L.n = xyz(d); L.before = d.w; L.le = xyz(e);
  return L;
}
__device__ __forceinline__ uint32_t pick_light(const DevScene& sc, float v1) {   // by area, on the value (frozen for the score)
  const float target = v1 * sc.light_total;
  uint32_t j = 0;
  while (j + 1 < sc.n_lights && !(target < __ldg(&sc.lights[5 * (size_t)j].w))) ++j;
  return j;
}

template <class T> struct VertexOut {
  V3<T> o2, d2;      // next ray
  T pb;              // density of d2 per solid angle (valid if pb_valid)
  T W[3];            // throughput factor of the direction sample
  T fcos[3], lw[3];  // emitter connection, per unit throughput, if it is visible: f_s cos  and  Le w_l / p_l  (C = fcos * lw)
  V3<T> y;           // the sampled point on the emitter
  bool pb_valid, alive, nee_valid;
};

// Emitter connection of a Lambert / GGX vertex at `hit` (Q21): fills out.nee_valid, out.y, out.fcos, out.lw and light_j.
// A function of (hit, v1, v2) -- and of d for a GGX vertex -- so that the score's reverse sweep can differentiate it on its own.
template <class T, bool NEE = true>
__device__ __forceinline__ void nee_connect(const DevScene& sc, const Frame& fr, float4 m0, float4 m1, uint32_t kind, V3<T> d, V3<T> hit,
                                            T v1, T v2, VertexOut<T>& out, uint32_t& light_j) {
  out.nee_valid = false;
  out.fcos[0] = out.fcos[1] = out.fcos[2] = out.lw[0] = out.lw[1] = out.lw[2] = lift_t<T>(0.f);
  // ---- next-event estimation at a Lambert / GGX vertex (Q21)
  if (NEE && sc.nee && kind != 1u && sc.n_lights) {
    const uint32_t j = pick_light(sc, val(v1));
    light_j = j;
    const Light L = load_light(sc, j);
    const T v1r = (v1 * sc.light_total - L.before) / L.area;
    const T su = sqrt_t(v1r);
    const T b1 = su * (1.0f - v2), b2 = su * v2;
    V3<T> y;
    y.x = (L.v0.x + L.e1.x * b1) + L.e2.x * b2; y.y = (L.v0.y + L.e1.y * b1) + L.e2.y * b2; y.z = (L.v0.z + L.e1.z * b1) + L.e2.z * b2;
    out.y = y;
    const V3<T> wv = vsub(y, hit);
    const T r2 = dott(wv, wv);
    const V3<T> w = vscale(wv, 1.0f / sqrt_t(r2));
    const T cos_x = dotf(w, fr.nf), cos_l = -dotf(w, L.n);
    if (val(cos_x) > 0.f && val(cos_l) > 0.f) {
      out.nee_valid = true;
      const T p_l = r2 / (cos_l * sc.light_total);
      T fcos[3], p_b;
      if (kind == 0u) {
        fcos[0] = cos_x * (m0.y * kInvPi); fcos[1] = cos_x * (m0.z * kInvPi); fcos[2] = cos_x * (m0.w * kInvPi);
        p_b = cos_x * kInvPi;
      } else {
        const float al = m1.y;
        V3<T> wo, wi;
        wo.x = -dotf(d, fr.t); wo.y = -dotf(d, fr.bf); wo.z = -dotf(d, fr.nf);
        wi.x = dotf(w, fr.t); wi.y = dotf(w, fr.bf); wi.z = cos_x;
        const V3<T> hm = vnormalize(vadd(wo, wi));
        const T woh = dott(wo, hm);
        const T c1 = 1.0f - woh;
        const T c5 = c1 * c1 * c1 * c1 * c1;
        const T Dh = ggx_d(hm, al);
        const T G1o = ggx_g1(wo, al), G1i = ggx_g1(wi, al);
        p_b = G1o * Dh / (wo.z * 4.0f);
        fcos[0] = (m0.y + (1.0f - m0.y) * c5) * G1i * p_b;
        fcos[1] = (m0.z + (1.0f - m0.z) * c5) * G1i * p_b;
        fcos[2] = (m0.w + (1.0f - m0.w) * c5) * G1i * p_b;
      }
      const T w_l = p_l / (p_l + p_b);
      out.fcos[0] = fcos[0]; out.fcos[1] = fcos[1]; out.fcos[2] = fcos[2];
      out.lw[0] = L.le.x * w_l / p_l; out.lw[1] = L.le.y * w_l / p_l; out.lw[2] = L.le.z * w_l / p_l;
    }
  }
}

// Direction sample of a GGX vertex: out.alive, out.d2, out.W and, with next-event estimation, the density out.pb of d2.
// A function of (d, u1, u2): the reverse sweep differentiates it on its own (out.alive / pb_valid / pb must come in cleared).
template <class T, bool NEE = true>
__device__ __forceinline__ void ggx_sample(const DevScene& sc, const Frame& fr, float4 m0, float4 m1, V3<T> d, T u1, T u2, VertexOut<T>& out) {
  T c5, G1;
  V3<T> hm;
  if (!ggx_dir<T>(fr, m1.y, d, u1, u2, out.d2, c5, G1, &hm)) {
    out.alive = false;
    out.W[0] = out.W[1] = out.W[2] = lift_t<T>(0.f);
    out.d2 = d;
  } else {
    out.W[0] = (m0.y + (1.0f - m0.y) * c5) * G1; out.W[1] = (m0.z + (1.0f - m0.z) * c5) * G1; out.W[2] = (m0.w + (1.0f - m0.w) * c5) * G1;
    if (NEE && sc.nee) {
      V3<T> wo;
      wo.x = -dotf(d, fr.t); wo.y = -dotf(d, fr.bf); wo.z = -dotf(d, fr.nf);
      out.pb_valid = true;
      out.pb = ggx_g1(wo, m1.y) * ggx_d(hm, m1.y) / (wo.z * 4.0f);
    }
  }
}

// hit: the point on the triangle's plane.  `decide`: take the lobe decision here (float instantiation) or use `reflect`.
template <class T, bool NEE = true>
__device__ __forceinline__ void vertex_fn(const DevScene& sc, float3 v0, const Frame& fr, float dn, float4 m0, float4 m1, uint32_t kind,
                                          V3<T> o, V3<T> d, T u1, T u2, T v1, T v2, bool decide, bool& reflect, VertexOut<T>& out,
                                          V3<T>& hit_out, uint32_t& light_j) {
  const float side = dn < 0.f ? 1.f : -1.f;
  const float3 n = fr.nf * side;   // the geometric normal again (exact: * +-1)
  // 1b: hit point on the frozen triangle's plane, t = ((v0 - o).n) / (d.n)
  const T tp = dotf(vsubf(v0, o), n) / dotf(d, n);
  V3<T> hit;
  hit.x = o.x + d.x * tp; hit.y = o.y + d.y * tp; hit.z = o.z + d.z * tp;
  hit_out = hit;
  nee_connect<T, NEE>(sc, fr, m0, m1, kind, d, hit, v1, v2, out, light_j);
  // ---- direction sample
  out.alive = true;
  out.pb_valid = false;
  out.pb = lift_t<T>(0.f);
  out.W[0] = out.W[1] = out.W[2] = lift_t<T>(1.f);
  float off = 1.f;
  if (kind == 0u) {
    out.d2 = lambert_dir<T>(fr, u1, u2);
    out.W[0] = lift_t<T>(m0.y); out.W[1] = lift_t<T>(m0.z); out.W[2] = lift_t<T>(m0.w);
    out.pb_valid = true;
    out.pb = sqrt_t(1.0f - u1) * kInvPi;
  } else if (kind == 1u) {
    const float eta = dn < 0.f ? m1.x : 1.0f / m1.x;
    if (decide) reflect = val(u1) < fresnel_dielectric(-dot3(make_float3(val(d.x), val(d.y), val(d.z)), fr.nf), eta);
    if (!reflect) off = -1.f;
    out.d2 = dielectric_dir<T>(fr, eta, reflect, d);
  } else {
    ggx_sample<T, NEE>(sc, fr, m0, m1, d, u1, u2, out);
  }
  const float k = sc.eps_ray * off;
  out.o2.x = hit.x + fr.nf.x * k; out.o2.y = hit.y + fr.nf.y * k; out.o2.z = hit.z + fr.nf.z * k;
}

// An emitter reached by the direction sample (front face): balance-heuristic weight against next-event estimation.
template <class T, bool NEE = true>
__device__ __forceinline__ T emitter_weight(const DevScene& sc, float3 v0, float3 n, V3<T> o, V3<T> d, T pb, bool pb_valid) {
  if (!(NEE && sc.nee && pb_valid)) return lift_t<T>(1.f);
  const T te = dotf(vsubf(v0, o), n) / dotf(d, n);
  const T p_l = (te * te) / ((-dotf(d, n)) * sc.light_total);
  return pb / (pb + p_l);
}

}  // namespace dr
