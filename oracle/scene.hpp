// TEST INFRASTRUCTURE — CPU oracle (see philox.hpp header).
//
// Triangle scene + closest-hit query.  The paper uses a hardware ray-tracing pipeline
// and never describes the acceleration structure; the oracle therefore
// implements the *definition* of a closest hit: brute force over all triangles with the
// DESIGN.md Q8 formula and tie rule.  A plain median-split BVH2 gives the same answer
// faster for the large scenes; tests/test_oracle_scene.py requires BVH2 == brute force
// bit for bit on seeded rays.
#pragma once
#include <algorithm>
#include <cstdint>
#include <limits>
#include <vector>

#include "dual.hpp"

namespace orc {

enum MatKind : int { MAT_LAMBERT = 0, MAT_DIELECTRIC = 1, MAT_GGX = 2, MAT_EMITTER = 3 };

template <class Real> struct Material {
  int kind;
  Real a[3];   // albedo (Lambert) or F0 (GGX conductor)
  Real ior;    // dielectric
  Real alpha;  // GGX roughness
  Real Le[3];  // emitter radiance (front face)
};

template <class Real> struct Hit {
  Real t;
  uint32_t tri;
  bool ok;
};

template <class Real> struct Scene {
  using V = Vec3<Real>;
  // geometry
  std::vector<V> v0, e1, e2;        // per triangle: vertex 0 and the two edges (v1-v0, v2-v0)
  std::vector<uint32_t> tri_mat;
  std::vector<Material<Real>> mats;
  Real env[3];
  // camera (Q4/1a): pinhole
  V cam_pos, cam_w, cam_r, cam_v;
  Real tan_half, aspect;
  uint32_t W, H, L;  // image size, max path length (segments); PSS dim d = 2L
  Real eps_ray;      // Q8: 1e-5 * bounding-box diagonal
  // analytic 2-D target instead of geometry (d = 2)
  bool analytic = false;
  std::vector<Real> mix_w, mix_mx, mix_my, mix_s;
  // BVH2 (median split)
  struct Node { V lo, hi; uint32_t left, right, first, count; };
  std::vector<Node> nodes;
  std::vector<uint32_t> order;  // triangle ids in leaf order
  bool use_bvh = true;

  // next-event estimation (Q21): the emitter triangles in index order with their areas and running sums
  bool nee = false;
  std::vector<uint32_t> light_tri;
  std::vector<Real> light_area, light_cdf;  // light_cdf[j] = area_0 + ... + area_j, summed in this order
  Real light_total = 0;

  void build_lights() {
    light_tri.clear(); light_area.clear(); light_cdf.clear(); light_total = 0;
    for (uint32_t t = 0; t < ntris(); ++t) {
      if (mats[tri_mat[t]].kind != MAT_EMITTER) continue;
      const V c = cross(e1[t], e2[t]);
      const Real a = Real(0.5) * std::sqrt(dot(c, c));
      if (!(a > Real(0)) || !std::isfinite(a)) continue;   // DESIGN.md Q21: an emitter without area is not on the list (sampling by area gives it probability zero)
      light_total = light_total + a;
      light_tri.push_back(t); light_area.push_back(a); light_cdf.push_back(light_total);
    }
    if (!(light_total > Real(0))) { light_tri.clear(); light_area.clear(); light_cdf.clear(); light_total = 0; }
  }

  uint32_t dim() const { return analytic ? 2u : (nee ? 4u : 2u) * L; }
  uint32_t ntris() const { return (uint32_t)v0.size(); }

  // Moeller-Trumbore, no culling, t_min = 0 exclusive (Q8).  Updates `best`
  // under the tie rule: smaller t, then smaller triangle index.
  inline void test_tri(uint32_t id, const V& o, const V& d, Hit<Real>& best) const {
    const V pv = cross(d, e2[id]);
    const Real det = dot(e1[id], pv);
    if (det == Real(0)) return;
    const Real inv = Real(1) / det;
    const V tv = o - v0[id];
    const Real u = dot(tv, pv) * inv;
    if (u < Real(0) || u > Real(1)) return;
    const V qv = cross(tv, e1[id]);
    const Real v = dot(d, qv) * inv;
    if (v < Real(0) || u + v > Real(1)) return;
    const Real t = dot(e2[id], qv) * inv;
    if (!(t > Real(0))) return;
    if (!best.ok || t < best.t || (t == best.t && id < best.tri)) {
      best.t = t; best.tri = id; best.ok = true;
    }
  }

  Hit<Real> intersect_brute(const V& o, const V& d) const {
    Hit<Real> best{std::numeric_limits<Real>::infinity(), 0u, false};
    for (uint32_t i = 0; i < ntris(); ++i) test_tri(i, o, d, best);
    return best;
  }

  static inline bool slab(const V& lo, const V& hi, const V& o, const V& inv, Real tbest) {
    Real tmin = Real(0), tmax = tbest;
    const Real lo_[3] = {lo.x, lo.y, lo.z}, hi_[3] = {hi.x, hi.y, hi.z};
    const Real o_[3] = {o.x, o.y, o.z}, i_[3] = {inv.x, inv.y, inv.z};
    for (int a = 0; a < 3; ++a) {
      Real t0 = (lo_[a] - o_[a]) * i_[a], t1 = (hi_[a] - o_[a]) * i_[a];
      if (t0 > t1) std::swap(t0, t1);
      // NaN (0 * inf) never narrows the interval
      if (t0 > tmin) tmin = t0;
      if (t1 < tmax) tmax = t1;
    }
    return tmin <= tmax;
  }

  Hit<Real> intersect_bvh(const V& o, const V& d) const {
    Hit<Real> best{std::numeric_limits<Real>::infinity(), 0u, false};
    if (nodes.empty()) return best;
    const V inv{Real(1) / d.x, Real(1) / d.y, Real(1) / d.z};
    uint32_t stack[128];
    int sp = 0;
    stack[sp++] = 0;
    while (sp) {
      const Node& n = nodes[stack[--sp]];
      if (!slab(n.lo, n.hi, o, inv, best.t)) continue;
      if (n.count) {
        for (uint32_t k = 0; k < n.count; ++k) test_tri(order[n.first + k], o, d, best);
      } else {
        stack[sp++] = n.left;
        stack[sp++] = n.right;
      }
    }
    return best;
  }

  Hit<Real> intersect(const V& o, const V& d) const { return use_bvh ? intersect_bvh(o, d) : intersect_brute(o, d); }

  // ---- construction -------------------------------------------------------------------
  void set_geometry(const float* verts, uint32_t nv, const uint32_t* idx, uint32_t nt) {
    (void)nv;
    v0.resize(nt); e1.resize(nt); e2.resize(nt);
    V lo{Real(1e30), Real(1e30), Real(1e30)}, hi{Real(-1e30), Real(-1e30), Real(-1e30)};
    auto vert = [&](uint32_t i) { return V{Real(verts[3 * i]), Real(verts[3 * i + 1]), Real(verts[3 * i + 2])}; };
    for (uint32_t t = 0; t < nt; ++t) {
      const V a = vert(idx[3 * t]), b = vert(idx[3 * t + 1]), c = vert(idx[3 * t + 2]);
      v0[t] = a; e1[t] = b - a; e2[t] = c - a;
      for (const V& p : {a, b, c}) {
        lo.x = std::min(lo.x, p.x); lo.y = std::min(lo.y, p.y); lo.z = std::min(lo.z, p.z);
        hi.x = std::max(hi.x, p.x); hi.y = std::max(hi.y, p.y); hi.z = std::max(hi.z, p.z);
      }
    }
    const V dg = hi - lo;
    const Real diag = std::sqrt(dot(dg, dg));
    eps_ray = Real(1e-5) * diag;
    build_bvh(Real(4e-6) * diag);
  }

  void set_camera(const float pos[3], const float look[3], const float up[3], float vfov_deg, uint32_t w, uint32_t h) {
    W = w; H = h;
    cam_pos = V{Real(pos[0]), Real(pos[1]), Real(pos[2])};
    const V lk{Real(look[0]), Real(look[1]), Real(look[2])}, u{Real(up[0]), Real(up[1]), Real(up[2])};
    cam_w = normalize(lk - cam_pos);
    cam_r = normalize(cross(cam_w, u));
    cam_v = cross(cam_r, cam_w);
    tan_half = std::tan(Real(vfov_deg) * Real(3.14159265358979323846 / 360.0));
    aspect = Real(W) / Real(H);
  }

 private:
  void build_bvh(Real pad) {
    const uint32_t nt = ntris();
    order.resize(nt);
    for (uint32_t i = 0; i < nt; ++i) order[i] = i;
    nodes.clear();
    if (!nt) return;
    nodes.reserve(2 * nt);
    std::vector<V> cen(nt);
    for (uint32_t i = 0; i < nt; ++i) cen[i] = v0[i] + (e1[i] + e2[i]) * Real(1.0 / 3.0);
    build_rec(0, nt, cen, pad);
  }
  uint32_t build_rec(uint32_t first, uint32_t count, const std::vector<V>& cen, Real pad) {
    const uint32_t me = (uint32_t)nodes.size();
    nodes.push_back(Node{});
    V lo{Real(1e30), Real(1e30), Real(1e30)}, hi{Real(-1e30), Real(-1e30), Real(-1e30)};
    V clo = lo, chi = hi;
    for (uint32_t k = first; k < first + count; ++k) {
      const uint32_t id = order[k];
      const V a = v0[id], b = v0[id] + e1[id], c = v0[id] + e2[id];
      for (const V& p : {a, b, c}) {
        lo.x = std::min(lo.x, p.x); lo.y = std::min(lo.y, p.y); lo.z = std::min(lo.z, p.z);
        hi.x = std::max(hi.x, p.x); hi.y = std::max(hi.y, p.y); hi.z = std::max(hi.z, p.z);
      }
      const V& cc = cen[id];
      clo.x = std::min(clo.x, cc.x); clo.y = std::min(clo.y, cc.y); clo.z = std::min(clo.z, cc.z);
      chi.x = std::max(chi.x, cc.x); chi.y = std::max(chi.y, cc.y); chi.z = std::max(chi.z, cc.z);
    }
    const V p{pad, pad, pad};
    nodes[me].lo = lo - p; nodes[me].hi = hi + p;
    nodes[me].first = first; nodes[me].count = count; nodes[me].left = nodes[me].right = 0;
    if (count <= 4) return me;
    const V ext = chi - clo;
    int axis = 0;
    if (ext.y > ext.x) axis = 1;
    if (ext.z > (axis == 0 ? ext.x : ext.y)) axis = 2;
    auto key = [&](uint32_t id) { return axis == 0 ? cen[id].x : (axis == 1 ? cen[id].y : cen[id].z); };
    const uint32_t mid = count / 2;
    std::nth_element(order.begin() + first, order.begin() + first + mid, order.begin() + first + count,
                     [&](uint32_t a, uint32_t b) { const Real ka = key(a), kb = key(b); return ka < kb || (ka == kb && a < b); });
    nodes[me].count = 0;
    const uint32_t l = build_rec(first, mid, cen, pad);
    const uint32_t r = build_rec(first + mid, count - mid, cen, pad);
    nodes[me].left = l; nodes[me].right = r;
    return me;
  }
};

}  // namespace orc
