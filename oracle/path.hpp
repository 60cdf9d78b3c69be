// TEST INFRASTRUCTURE — CPU oracle (see philox.hpp header).
//
// Target evaluation x -> (f, p, pixelIndex, score): the integrand f(x), the target
// density p = luminance(f) ("e.g., luminance"), the pixel "hit by
// state.x[0]" (Alg. 1) and score = grad ln(p + eps), eps = 1e-8
// (Alg. 4 line 1 L710).  The paper never describes its path sampling
// routines; what follows is the DESIGN.md reading Q4-Q9, step by step.
// With next-event estimation (scene flag `nee`, Q21; "same underlying path sampling routines",
// L757 "MCMC sampling for both direct and indirect illumination") every vertex owns four coordinates, x[4k..4k+3] =
// (u1, u2: direction sample; v1, v2: point on the emitters), d = 4L, and x[2], x[3] are unused.  At a Lambert or GGX
// vertex the emitters are sampled uniformly by area, the connection is weighted against the direction sample by the
// balance heuristic (Veach 1995), and an emitter found by the direction sample carries the complementary weight.
// The same template runs with S = Real (values only) and S = Dual<Real, D> (values and
// d/dx of everything, discrete decisions frozen on the value part = what AD computes).
#pragma once
#include <cmath>
#include <cstdint>

#include "scene.hpp"

namespace orc {

constexpr double kEps = 1e-8;
constexpr double kLumR = 0.2126, kLumG = 0.7152, kLumB = 0.0722;
constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr double kPi = 3.1415926535897932384626433832795;
constexpr double kInvPi = 0.31830988618379067153776752674503;

template <class S> struct PathOut {
  S f[3];
  S p;
  uint32_t pix;
  uint32_t nrays;
  uint32_t sig;  // FNV-1a hash of the discrete decisions (triangle per segment, lobe per vertex)
};

inline uint32_t fnv(uint32_t h, uint32_t v) { return (h ^ v) * 16777619u; }

// Pixel of a PSS point (Q4): px = min(floor(x0 W), W-1), py = min(floor(x1 H), H-1), row 0 on top.
template <class Real> inline uint32_t pixel_of(Real x0, Real x1, uint32_t W, uint32_t H) {
  uint32_t px = (uint32_t)std::floor(x0 * Real(W)), py = (uint32_t)std::floor(x1 * Real(H));
  if (px > W - 1) px = W - 1;
  if (py > H - 1) py = H - 1;
  return py * W + px;
}

// Exact unpolarised Fresnel reflectance for a smooth dielectric (Q7); eta = n_t / n_i.
template <class Real> inline Real fresnel_dielectric(Real cos_i, Real eta, Real& cos_t) {
  const Real sin2_t = (Real(1) - cos_i * cos_i) / (eta * eta);
  if (sin2_t >= Real(1)) { cos_t = Real(0); return Real(1); }  // total internal reflection
  cos_t = std::sqrt(Real(1) - sin2_t);
  const Real r_par = (eta * cos_i - cos_t) / (eta * cos_i + cos_t);
  const Real r_perp = (cos_i - eta * cos_t) / (cos_i + eta * cos_t);
  return Real(0.5) * (r_par * r_par + r_perp * r_perp);
}

// x: d = 2L coordinates in [0,1).  Mesh scenes only (analytic targets: analytic2d.hpp).
template <class Real, class S> void eval_path(const Scene<Real>& sc, const S* x, PathOut<S>& out) {
  using VS = Vec3<S>;
  using VR = Vec3<Real>;
  using orc::sqrt; using orc::sin; using orc::cos;
  const uint32_t L = sc.L;
  out.f[0] = out.f[1] = out.f[2] = S(Real(0));
  out.pix = pixel_of<Real>(value(x[0]), value(x[1]), sc.W, sc.H);
  out.nrays = 0;
  uint32_t sig = 2166136261u;

  // 1a. camera ray through the film point (x0 W, x1 H)
  const S sx = (Real(2) * x[0] - Real(1)) * (sc.tan_half * sc.aspect);
  const S sy = (Real(2) * x[1] - Real(1)) * sc.tan_half;
  VS d = normalize(lift<S>(sc.cam_w) + lift<S>(sc.cam_r) * sx - lift<S>(sc.cam_v) * sy);
  VS o = lift<S>(sc.cam_pos);
  S T[3] = {S(Real(1)), S(Real(1)), S(Real(1))};
  const uint32_t stride = sc.nee ? 4u : 2u;   // coordinates per vertex
  bool pb_valid = false;                       // the last direction came from a sampler with a density (Lambert, GGX)
  S pb = S(Real(0));                           // that density, per solid angle

  for (uint32_t k = 1; k <= L; ++k) {
    const VR ov{value(o.x), value(o.y), value(o.z)}, dv{value(d.x), value(d.y), value(d.z)};
    const Hit<Real> h = sc.intersect(ov, dv);
    ++out.nrays;
    if (!h.ok) {  // escaped: environment radiance
      sig = fnv(sig, 0u);
      for (int c = 0; c < 3; ++c) out.f[c] = out.f[c] + T[c] * sc.env[c];
      break;
    }
    sig = fnv(sig, h.tri + 1u);
    const Material<Real>& m = sc.mats[sc.tri_mat[h.tri]];
    // geometric frame of the frozen triangle (Q6)
    const VR e1 = sc.e1[h.tri], e2 = sc.e2[h.tri];
    const VR tg = normalize(e1);
    const VR n = normalize(cross(e1, e2));
    const VR bt = cross(n, tg);
    const Real dn = dot(dv, n);
    if (m.kind == MAT_EMITTER) {  // DiffuseAreaLight-like: front face emits, path always stops
      if (dn < Real(0)) {
        sig = fnv(sig, 4u);
        S w_b = S(Real(1));   // balance-heuristic weight of the direction sample against next-event estimation
        if (sc.nee && pb_valid) {
          const VS nS = lift<S>(n);
          const S te = dot(lift<S>(sc.v0[h.tri]) - o, nS) / dot(d, nS);      // distance to the emitter's plane
          const S p_l = (te * te) / ((-dot(d, nS)) * sc.light_total);         // area density 1 / total -> solid angle
          w_b = pb / (pb + p_l);
        }
        for (int c = 0; c < 3; ++c) out.f[c] = out.f[c] + T[c] * m.Le[c] * w_b;
      } else {
        sig = fnv(sig, 5u);
      }
      break;
    }
    if (k == L) break;  // length cap: no further vertex to sample
    // 1b. hit point on the frozen triangle's plane: t = ((v0 - o).n) / (d.n)
    const VS nS = lift<S>(n);
    const S t = dot(lift<S>(sc.v0[h.tri]) - o, nS) / dot(d, nS);
    const VS hit = o + d * t;
    const Real side = dn < Real(0) ? Real(1) : Real(-1);  // n_f = side * n faces the incoming ray
    const VS nf = lift<S>(n * side), bf = lift<S>(bt * side), tS = lift<S>(tg);
    const S u1 = x[stride * k], u2 = x[stride * k + 1];
    VS dnew;
    Real off_side = Real(1);  // +1: leave on the n_f side, -1: on the far side
    // ---- next-event estimation at a Lambert / GGX vertex (Q21)
    if (sc.nee && m.kind != MAT_DIELECTRIC && !sc.light_tri.empty()) {
      const S v1 = x[stride * k + 2], v2 = x[stride * k + 3];
      // emitter triangle by area (frozen on the value), then a uniform point on it
      const Real target = value(v1) * sc.light_total;
      uint32_t j = 0;
      while (j + 1 < sc.light_tri.size() && !(target < sc.light_cdf[j])) ++j;
      const Real before = j ? sc.light_cdf[j - 1] : Real(0);
      const S v1r = (v1 * sc.light_total - before) / sc.light_area[j];
      const S su = sqrt(v1r);
      const uint32_t lt = sc.light_tri[j];
      const VS y = lift<S>(sc.v0[lt]) + lift<S>(sc.e1[lt]) * (su * (Real(1) - v2)) + lift<S>(sc.e2[lt]) * (su * v2);
      const VS wv = y - hit;
      const S r2 = dot(wv, wv);
      const VS w = wv * (Real(1) / sqrt(r2));
      const VR nl = normalize(cross(sc.e1[lt], sc.e2[lt]));
      const S cos_x = dot(w, nf), cos_l = -dot(w, lift<S>(nl));
      if (value(cos_x) > Real(0) && value(cos_l) > Real(0)) {
        const S p_l = r2 / (cos_l * sc.light_total);
        S fcos[3], p_b;
        if (m.kind == MAT_LAMBERT) {
          for (int c = 0; c < 3; ++c) fcos[c] = cos_x * (m.a[c] * Real(kInvPi));
          p_b = cos_x * Real(kInvPi);
        } else {  // GGX conductor: F D G1(wo) G1(wi) / (4 cos_o), density of the visible-normal sampler G1(wo) D / (4 cos_o)
          const Real al = m.alpha;
          const VS wo{-dot(d, tS), -dot(d, bf), -dot(d, nf)};
          const VS wi{dot(w, tS), dot(w, bf), cos_x};
          const VS hm = normalize(wo + wi);
          const S woh = dot(wo, hm);
          const S c1 = Real(1) - woh;
          const S c5 = c1 * c1 * c1 * c1 * c1;
          const S q = hm.z * hm.z * (al * al - Real(1)) + Real(1);
          const S Dh = (al * al * Real(kInvPi)) / (q * q);
          const S G1o = (Real(2) * wo.z) / (wo.z + sqrt((wo.x * wo.x + wo.y * wo.y) * (al * al) + wo.z * wo.z));
          const S G1i = (Real(2) * wi.z) / (wi.z + sqrt((wi.x * wi.x + wi.y * wi.y) * (al * al) + wi.z * wi.z));
          p_b = G1o * Dh / (Real(4) * wo.z);
          for (int c = 0; c < 3; ++c) fcos[c] = (m.a[c] + (Real(1) - m.a[c]) * c5) * G1i * p_b;
        }
        // visibility: the closest hit from the offset point towards y is that emitter triangle (a decision, on values)
        const VS os = hit + nf * S(sc.eps_ray);
        const VR osv{value(os.x), value(os.y), value(os.z)};
        const VR dsv = normalize(VR{value(y.x), value(y.y), value(y.z)} - osv);
        const Hit<Real> hs = sc.intersect(osv, dsv);
        ++out.nrays;
        const bool vis = hs.ok && hs.tri == lt;
        sig = fnv(sig, vis ? 7u : 6u);
        if (vis) {
          const S w_l = p_l / (p_l + p_b);
          const Material<Real>& ml = sc.mats[sc.tri_mat[lt]];
          for (int c = 0; c < 3; ++c) out.f[c] = out.f[c] + T[c] * fcos[c] * (ml.Le[c] * w_l / p_l);
        }
      }
    }
    if (m.kind == MAT_LAMBERT) {
      sig = fnv(sig, 0u);
      const S r = sqrt(u1), phi = Real(kTwoPi) * u2;
      const S wx = r * cos(phi), wy = r * sin(phi), wz = sqrt(Real(1) - u1);
      dnew = tS * wx + bf * wy + nf * wz;
      for (int c = 0; c < 3; ++c) T[c] = T[c] * m.a[c];
      pb_valid = true; pb = wz * Real(kInvPi);
    } else if (m.kind == MAT_DIELECTRIC) {
      // entering (d.n < 0): eta = ior / 1; leaving: eta = 1 / ior
      const Real eta = dn < Real(0) ? m.ior : Real(1) / m.ior;
      const S cos_i = -dot(d, nf);
      Real cos_t;
      const Real F = fresnel_dielectric<Real>(value(cos_i), eta, cos_t);
      if (value(u1) < F) {  // reflect (also total internal reflection, F = 1)
        sig = fnv(sig, 1u);
        dnew = d + nf * (Real(2) * cos_i);
      } else {              // refract
        sig = fnv(sig, 2u);
        const S ct = sqrt(Real(1) - (Real(1) - cos_i * cos_i) / (eta * eta));
        dnew = d * S(Real(1) / eta) + nf * (cos_i / eta - ct);
        off_side = Real(-1);
      }
      pb_valid = false;  // a Dirac lobe: next-event estimation cannot produce this path
      // weight 1 for both lobes (Q7)
    } else {  // MAT_GGX: conductor, visible-normal sampling (spherical-cap form), Q7
      sig = fnv(sig, 3u);
      const Real al = m.alpha;
      const VS wo{-dot(d, tS), -dot(d, bf), -dot(d, nf)};
      const VS ws = normalize(VS{wo.x * al, wo.y * al, wo.z});
      const S phi = Real(kTwoPi) * u2;
      const S z = (Real(1) - u1) * (Real(1) + ws.z) - ws.z;
      S s2 = Real(1) - z * z;
      if (value(s2) < Real(0)) s2 = S(Real(0));
      const S st = sqrt(s2);
      const VS hs{st * cos(phi) + ws.x, st * sin(phi) + ws.y, z + ws.z};
      const VS hm = normalize(VS{hs.x * al, hs.y * al, hs.z});
      const S woh = dot(wo, hm);
      const VS wi = hm * (Real(2) * woh) - wo;
      if (!(value(wi.z) > Real(0))) {  // below the horizon: weight 0, path ends
        T[0] = T[1] = T[2] = S(Real(0));
      } else {
        const S c1 = Real(1) - woh;
        const S c5 = c1 * c1 * c1 * c1 * c1;
        const S G1 = (Real(2) * wi.z) / (wi.z + sqrt((wi.x * wi.x + wi.y * wi.y) * (al * al) + wi.z * wi.z));
        for (int c = 0; c < 3; ++c) T[c] = T[c] * ((m.a[c] + (Real(1) - m.a[c]) * c5) * G1);
        dnew = tS * wi.x + bf * wi.y + nf * wi.z;
        if (sc.nee) {  // density of this direction: G1(wo) D(h) / (4 cos_o)
          const S q = hm.z * hm.z * (al * al - Real(1)) + Real(1);
          const S Dh = (al * al * Real(kInvPi)) / (q * q);
          const S G1o = (Real(2) * wo.z) / (wo.z + sqrt((wo.x * wo.x + wo.y * wo.y) * (al * al) + wo.z * wo.z));
          pb_valid = true; pb = G1o * Dh / (Real(4) * wo.z);
        }
      }
    }
    if (value(T[0]) == Real(0) && value(T[1]) == Real(0) && value(T[2]) == Real(0)) break;
    o = hit + nf * S(sc.eps_ray * off_side);
    d = dnew;
  }
  out.p = out.f[0] * Real(kLumR) + out.f[1] * Real(kLumG) + out.f[2] * Real(kLumB);
  out.sig = sig;
}

}  // namespace orc
