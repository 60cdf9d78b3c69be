// TEST INFRASTRUCTURE — CPU oracle (see philox.hpp header).
//
// Appendix C of the paper (Eq. "adjoint-bias" L456-L460): the field that controls the bias of the
// modified killing rate, b(y) = (L^* p_hat)(y) / p_hat(y), for the local dynamics of Alg. 4 seen as a jump process with
// holding rate lambda = 1 / dt (L659) and transition kernel K(x, .) = law of wrap(x + (s^2/2) g(x) + c~ rot(g(x)) + s xi):
//     (L^* p)(y) = lambda * ( integral p(x) k(x, y) dx - p(y) ),
//     k(x, y) = prod_i sum_j phi((y_i - m_i(x) + j) / s) / s,   m(x) = x + (s^2/2) g(x) + c~ (g_2(x), -g_1(x)),
// on the 2-D analytic target (analytic2d.hpp), g = grad p / (p + eps).  The integral is a midpoint rule on an M x M grid,
// written out as the double loop it is.  out[iy * G + ix] = b at the centre of cell (ix, iy) of a G x G grid.
#pragma once
#include <cmath>
#include <vector>

#include "analytic2d.hpp"

namespace orc {

template <class Real>
void bias_field(const Scene<Real>& sc, Real s, Real c_tilde, Real dt, uint32_t G, uint32_t M, double* out) {
  const Real lambda = Real(1) / dt, h = Real(0.5) * s * s;
  std::vector<Real> px((size_t)M * M), mx((size_t)M * M), my((size_t)M * M);
  for (uint32_t j = 0; j < M; ++j)
    for (uint32_t i = 0; i < M; ++i) {
      const Real x0 = (Real(i) + Real(0.5)) / Real(M), x1 = (Real(j) + Real(0.5)) / Real(M);
      Real p, gx, gy;
      eval_analytic<Real>(sc, x0, x1, p, gx, gy);
      const Real g0 = gx / (p + Real(kEps)), g1 = gy / (p + Real(kEps));
      px[(size_t)j * M + i] = p;
      mx[(size_t)j * M + i] = x0 + h * g0 + c_tilde * g1;     // Alg. 4 lines 2-4 without the noise
      my[(size_t)j * M + i] = x1 + h * g1 - c_tilde * g0;
    }
  const Real norm = Real(0.3989422804014326779399460599343) / s;
#pragma omp parallel for schedule(dynamic, 4)
  for (int64_t c = 0; c < (int64_t)G * G; ++c) {
    const Real y0 = (Real(c % G) + Real(0.5)) / Real(G), y1 = (Real(c / G) + Real(0.5)) / Real(G);
    double acc = 0;
    for (size_t k = 0; k < (size_t)M * M; ++k) {
      const Real d0 = min_image<Real>(y0 - mx[k]), d1 = min_image<Real>(y1 - my[k]);
      Real w0 = 0, w1 = 0;
      for (int j = -1; j <= 1; ++j) {   // wrapped Gaussian: the nearest images (s << 1)
        const Real z0 = (d0 + Real(j)) / s, z1 = (d1 + Real(j)) / s;
        w0 += norm * std::exp(Real(-0.5) * z0 * z0);
        w1 += norm * std::exp(Real(-0.5) * z1 * z1);
      }
      acc += (double)(px[k] * w0 * w1);
    }
    acc /= (double)M * (double)M;
    Real p, gx, gy;
    eval_analytic<Real>(sc, y0, y1, p, gx, gy);
    out[c] = (double)lambda * (acc - (double)p) / (double)p;
  }
}

}  // namespace orc
