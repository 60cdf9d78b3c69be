// TEST INFRASTRUCTURE — CPU oracle (see philox.hpp header).
//
// 2-D analytic target with known normalisation: a mixture of wrapped Gaussians on the
// torus T^2 (the "Gaussian mode of an example target density" of PAPER.md L586-L640,
// used for the stationarity pins).  p(x) = sum_k w_k prod_{i<2} Wg(delta_i; s_k),
// Wg(delta; s) = sum_{j=-2..2} phi((delta + j) / s) / s, delta = minimal-image offset
// x_i - mu_i in [-0.5, 0.5).  Integral over T^2 = sum_k w_k (truncation error < 1e-40
// for s <= 0.15).  f = (p, p, p); score = grad p / (p + eps) in closed form.
#pragma once
#include <cmath>

#include "path.hpp"

namespace orc {

template <class Real> inline Real min_image(Real v) { return v - std::floor(v + Real(0.5)); }  // [-0.5, 0.5), tie -> -0.5

template <class Real> inline void wrapped_gauss(Real delta, Real s, Real& w, Real& dw) {
  w = 0; dw = 0;
  const Real inv = Real(1) / s, norm = Real(0.3989422804014326779399460599343) * inv;
  for (int j = -2; j <= 2; ++j) {
    const Real z = (delta + Real(j)) * inv;
    const Real e = norm * std::exp(Real(-0.5) * z * z);
    w += e;
    dw += -z * inv * e;
  }
}

// Returns p and grad p (not yet divided by p + eps).
template <class Real> inline void eval_analytic(const Scene<Real>& sc, Real x0, Real x1, Real& p, Real& gx, Real& gy) {
  p = 0; gx = 0; gy = 0;
  for (size_t k = 0; k < sc.mix_w.size(); ++k) {
    Real wx, dwx, wy, dwy;
    wrapped_gauss<Real>(min_image<Real>(x0 - sc.mix_mx[k]), sc.mix_s[k], wx, dwx);
    wrapped_gauss<Real>(min_image<Real>(x1 - sc.mix_my[k]), sc.mix_s[k], wy, dwy);
    p += sc.mix_w[k] * wx * wy;
    gx += sc.mix_w[k] * dwx * wy;
    gy += sc.mix_w[k] * wx * dwy;
  }
}

}  // namespace orc
