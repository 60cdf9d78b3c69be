// TEST INFRASTRUCTURE — CPU oracle (see philox.hpp header).
//
// The five samplers, one chain-iteration at a time, in the paper's order and notation:
//   Alg. 1 Initialize + Accumulate, Alg. 2 Evolve (L530-L543),
//   Alg. 3 Resolve (L545-L550), Alg. 4 LocalDynamics (L707-L723);
//   Metropolis / MALA local dynamics and the plain-MH estimator as read in DESIGN.md
//   Q11 (PAPER.md L733-L747 defers them to prior work);
//   lambda = 1/dt (L658-L659), kappa = kappa0 / p_hat (L443-L445 with uniform rho),
//   kappa0 = p_lambda / (m dt) (L750-L753), lambda == 1 for Metropolis-/MALA-Restore (L737).
// No blocking, fusion or reordering: a loop over chains, each doing exactly what the
// pseudocode says.  The only parallelism is OpenMP over chains for the target
// evaluation; decisions and accumulation run in chain order, so results do not depend
// on the thread count.
#pragma once
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

#include "analytic2d.hpp"
#include "path.hpp"
#include "philox.hpp"

namespace orc {

enum Method : int { METROPOLIS = 0, MALA = 1, METROPOLIS_RESTORE = 2, MALA_RESTORE = 3, DIFFUSION_RESTORE = 4,
                    PATH_TRACING = 5 };  // 5: ordinary path tracing on the same buffers: the baseline of section 6

struct Config {
  int method;
  uint32_t n_chains;
  double stddev;            // 1e-2 (Metropolis*), 5e-3 (Langevin-based)
  double c_tilde;           // rotation strength c~ = dt c / 2 (L700); value is DESIGN.md Q10
  double dt;                // L755: 1e-5 (Diffusion Restore)
  double m;                 // L754: 64
  double large_step_prob;   // L747: 0.3 (plain Metropolis / MALA only)
  double p_lambda_override; // <= 0: bootstrap from the init states (Q-a0)
  uint64_t seed;
  uint32_t chain_offset;    // global id of chain 0 (chains are keyed by global id: sharding-invariant, section 8e)
  int rao_blackwell;        // Restore variants: accumulate E[dtau | x] = 1 / (lambda + kappa) instead of the sampled dtau
                            // (Rao-Blackwellisation of the holding time; DESIGN.md f3)
  int a_mode = 0;           // antisymmetric part of the drift (L567, L687-L692, future work L822): 0 = the paper's
                            // diag(A_block): coordinate pairs (2i, 2i+1); 1 = pairs (4i, 4i+2), (4i+1, 4i+3): the two
                            // 2-blocks of a group of four rotate into each other (Q24)
  // Non-uniform regeneration density rho (L424-L430, L443-L445, future work L824; Q24): piecewise constant on a
  // rho_grid x rho_grid tiling of the film coordinates (x0, x1), uniform in every other coordinate.  rho_w: tile
  // probabilities, row-major (tile = ty * G + tx), summing to one, so rho = G^2 w[tile] and rho_lambda = 1.
  uint32_t rho_grid = 0;
  std::vector<double> rho_w;
};

template <class Real> struct Eval {
  Real f[3];
  Real p;
  uint32_t pix, nrays, sig;
  bool nonfinite;
};

// Toroidal wrap, Alg. 4 line 5 (L714): x -= floor(x); clamped below 1 (Q3).
template <class Real> inline Real wrap01(Real v) {
  const Real w = v - std::floor(v);
  const Real top = std::nextafter(Real(1), Real(0));
  return w < top ? w : top;
}

template <class Real, int D> inline void evaluate_dual(const Scene<Real>& sc, const Real* x, Eval<Real>& e, Real* g) {
  using Du = Dual<Real, D>;
  const uint32_t d = sc.dim();
  Du xs[D];
  for (uint32_t j = 0; j < d; ++j) xs[j] = Du::variable(x[j], (int)j);
  PathOut<Du> out;
  eval_path<Real, Du>(sc, xs, out);
  for (int c = 0; c < 3; ++c) e.f[c] = out.f[c].v;
  e.p = out.p.v; e.pix = out.pix; e.nrays = out.nrays; e.sig = out.sig;
  const Real denom = out.p.v + Real(kEps);  // score = grad p / (p + eps), L569
  for (uint32_t j = 0; j < d; ++j) g[j] = out.p.d[j] / denom;
}

// Target evaluation at x.  g (d entries) is written iff want_score.
template <class Real> inline void evaluate(const Scene<Real>& sc, const Real* x, bool want_score, Eval<Real>& e, Real* g) {
  const uint32_t d = sc.dim();
  e.nonfinite = false;
  if (sc.analytic) {
    Real p, gx, gy;
    eval_analytic<Real>(sc, x[0], x[1], p, gx, gy);
    e.f[0] = e.f[1] = e.f[2] = p; e.p = p;
    e.pix = pixel_of<Real>(x[0], x[1], sc.W, sc.H);
    e.nrays = 0; e.sig = 0;
    if (want_score) { g[0] = gx / (p + Real(kEps)); g[1] = gy / (p + Real(kEps)); }
  } else if (!want_score) {
    PathOut<Real> out;
    eval_path<Real, Real>(sc, x, out);
    for (int c = 0; c < 3; ++c) e.f[c] = out.f[c];
    e.p = out.p; e.pix = out.pix; e.nrays = out.nrays; e.sig = out.sig;
  } else if (d <= 4) evaluate_dual<Real, 4>(sc, x, e, g);
  else if (d <= 8) evaluate_dual<Real, 8>(sc, x, e, g);
  else if (d <= 16) evaluate_dual<Real, 16>(sc, x, e, g);
  else if (d <= 24) evaluate_dual<Real, 24>(sc, x, e, g);
  else if (d <= 32) evaluate_dual<Real, 32>(sc, x, e, g);
  else if (d <= 48) evaluate_dual<Real, 48>(sc, x, e, g);
  else evaluate_dual<Real, 64>(sc, x, e, g);
  // Q18: a non-finite contribution or score is a zero-contribution state, counted.
  bool bad = !(std::isfinite(e.f[0]) && std::isfinite(e.f[1]) && std::isfinite(e.f[2]) && std::isfinite(e.p));
  if (want_score) for (uint32_t j = 0; j < d; ++j) bad = bad || !std::isfinite(g[j]);
  if (bad) {
    e.nonfinite = true;
    e.f[0] = e.f[1] = e.f[2] = e.p = 0;
    if (want_score) for (uint32_t j = 0; j < d; ++j) g[j] = 0;
  }
}

template <class Real> struct Chains {
  const Scene<Real>& sc;
  Config cfg;
  uint32_t N, d, npix;
  bool restore, grad;
  // state record of PAPER.md L468-L480 (rng replaced by counter-based keying, Q14) + cached score
  std::vector<Real> x, g, p, fop;  // N*d, N*d, N, N*3
  std::vector<uint32_t> pix, sig;
  std::vector<uint8_t> killed;
  // per-chain record of the last step's decisions (diagnostics for the parity harness)
  std::vector<uint8_t> accepted;   // 1 = proposal accepted / regenerated / Langevin move, 0 = rejected
  std::vector<Real> dtau;
  // buffers of PAPER.md L482-L493
  std::vector<double> accum;       // npix * 4: sum w f/p_hat (RGB), sum w / p_hat
  uint64_t tours = 0, mutations = 0, rays = 0, mh_accepts = 0, nonfinite = 0;
  uint32_t kills_last = 0;
  Real p_lambda = 0, kappa0 = 0, lambda = 1;
  uint32_t iteration = 0, epoch = 0;
  std::vector<uint32_t> queue;     // killed chain ids, ascending (Q13)

  Chains(const Scene<Real>& s, const Config& c) : sc(s), cfg(c) {
    N = c.n_chains; d = s.dim(); npix = s.W * s.H;
    restore = c.method >= METROPOLIS_RESTORE && c.method <= DIFFUSION_RESTORE;
    grad = c.method == MALA || c.method == MALA_RESTORE || c.method == DIFFUSION_RESTORE;
    x.assign((size_t)N * d, 0); g.assign((size_t)N * d, 0); p.assign(N, 0); fop.assign((size_t)N * 3, 0);
    pix.assign(N, 0); sig.assign(N, 0); killed.assign(N, 0); accepted.assign(N, 0); dtau.assign(N, 0);
    accum.assign((size_t)npix * 4, 0.0);
  }

  void uniform_point(uint32_t chain, uint32_t iter, uint32_t purpose, Real* y) const {
    for (uint32_t j = 0; j < d; j += 4) {
      uint32_t w[4];
      stream_block(cfg.seed, cfg.chain_offset + chain, iter, j / 4, purpose, epoch, w);
      for (uint32_t c = 0; c < 4 && j + c < d; ++c) y[j + c] = u01_co<Real>(w[c]);
    }
  }

  // ---- regeneration density rho (Q24) ----------------------------------------------------------------------------
  std::vector<Real> rho_w, rho_cdf;   // tile probabilities and their running sums, in the chains' precision
  void set_rho() {
    rho_w.clear(); rho_cdf.clear();
    Real acc = 0;
    for (double w : cfg.rho_w) { rho_w.push_back((Real)w); acc = acc + (Real)w; rho_cdf.push_back(acc); }
  }
  // x ~ rho from a uniform point: the tile by inversion of the running sums with y0, uniform inside the tile
  void regeneration_point(Real* y) const {
    const uint32_t G = cfg.rho_grid;
    if (!G) return;
    const Real u0 = y[0], u1 = y[1];
    uint32_t t = 0;
    while (t + 1 < G * G && !(u0 < rho_cdf[t])) ++t;
    const Real before = t ? rho_cdf[t - 1] : Real(0);
    const Real frac = (u0 - before) / rho_w[t];
    y[0] = wrap01<Real>((Real(t % G) + frac) / Real(G));
    y[1] = wrap01<Real>((Real(t / G) + u1) / Real(G));
  }
  Real rho_at(const Real* xx) const {   // rho / rho_lambda at a state
    const uint32_t G = cfg.rho_grid;
    if (!G) return Real(1);
    uint32_t tx = (uint32_t)std::floor(xx[0] * Real(G)), ty = (uint32_t)std::floor(xx[1] * Real(G));
    if (tx > G - 1) tx = G - 1;
    if (ty > G - 1) ty = G - 1;
    return Real(G) * Real(G) * rho_w[ty * G + tx];
  }
  void normals(uint32_t chain, uint32_t iter, Real* xi) const {
    for (uint32_t j = 0; j < d; j += 4) {
      uint32_t w[4];
      stream_block(cfg.seed, cfg.chain_offset + chain, iter, j / 4, PROP_N, epoch, w);
      Real z[4];
      box_muller<Real>(w[0], w[1], z[0], z[1]);
      box_muller<Real>(w[2], w[3], z[2], z[3]);
      for (uint32_t c = 0; c < 4 && j + c < d; ++c) xi[j + c] = z[c];
    }
  }

  void store(uint32_t i, const Real* y, const Eval<Real>& e, const Real* gy) {
    std::memcpy(&x[(size_t)i * d], y, d * sizeof(Real));
    if (grad) std::memcpy(&g[(size_t)i * d], gy, d * sizeof(Real));
    p[i] = e.p; pix[i] = e.pix; sig[i] = e.sig;
    const Real phat = e.p + Real(kEps);
    for (int c = 0; c < 3; ++c) fop[(size_t)i * 3 + c] = e.f[c] / phat;  // f / p_hat, Alg. 1 L523 with Q9
    if (cfg.method == PATH_TRACING) for (int c = 0; c < 3; ++c) fop[(size_t)i * 3 + c] = e.f[c];  // independent samples: f itself
  }

  // Accumulate, Alg. 1 L506-L526.  The target was evaluated when the state was stored.
  void accumulate(uint32_t i, uint32_t n) {
    uint32_t w[4];
    stream_block(cfg.seed, cfg.chain_offset + i, n, 0, DECIDE, epoch, w);
    const Real phat = p[i] + Real(kEps);
    Real weight = Real(1);
    if (restore) {
      const Real kappa = rho_at(&x[(size_t)i * d]) * kappa0 / phat;   // L445: (rho / rho_lambda) kappa0 / p_hat; uniform rho: 1 (L452)
      const Real dt1 = -std::log(u01_oc<Real>(w[2])) / lambda; // L511
      const Real dt2 = -std::log(u01_oc<Real>(w[3])) / kappa;  // L512
      if (dt1 < dt2) { weight = dt1; killed[i] = 0; }          // L513-L515
      else { weight = dt2; killed[i] = 1; ++tours; ++kills_last; }  // L516-L519 (tie -> killed, Q16)
      if (cfg.rao_blackwell) weight = Real(1) / (lambda + kappa);    // E[min(dt1, dt2)]; the kill decision stays the sampled race
    }
    dtau[i] = weight;
    ++mutations;
    if (p[i] > Real(0)) {                                      // L522
      double* a = &accum[(size_t)pix[i] * 4];
      for (int c = 0; c < 3; ++c) a[c] += (double)(weight * fop[(size_t)i * 3 + c]);  // L524
      a[3] += cfg.method == PATH_TRACING ? 1.0 : (double)(weight / phat);   // ratio-image denominator (Q12); PT: sample count
    }
  }

  void bootstrap() {
    if (cfg.p_lambda_override > 0) p_lambda = (Real)cfg.p_lambda_override;
    else {
      double s = 0;
      for (uint32_t i = 0; i < N; ++i) s += (double)(p[i] / rho_at(&x[(size_t)i * d]));   // init states are rho-distributed
      p_lambda = (Real)(s / (double)N + kEps);                 // normalisation of p_hat = p + eps
    }
    const Real dt_eff = cfg.method == DIFFUSION_RESTORE ? (Real)cfg.dt : Real(1);
    lambda = Real(1) / dt_eff;                                 // L659; == 1 for the MH-Restore variants (L737)
    kappa0 = p_lambda / ((Real)cfg.m * dt_eff);                // L752
  }

  // Alg. 1: x ~ nu (uniform, L687), evaluate, [bootstrap p_lambda, kappa0], Accumulate.
  void init(uint32_t frame) {
    epoch = frame; iteration = 0;
    set_rho();
    std::fill(accum.begin(), accum.end(), 0.0);
    tours = mutations = rays = mh_accepts = nonfinite = 0; kills_last = 0;
    std::vector<uint32_t> nr(N); std::vector<uint8_t> nf(N);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t ii = 0; ii < (int64_t)N; ++ii) {
      const uint32_t i = (uint32_t)ii;
      std::vector<Real> y(d), gy(d);
      uniform_point(i, 0, REGEN_U, y.data());
      regeneration_point(y.data());                            // x ~ nu = rho (Alg. 1)
      Eval<Real> e;
      evaluate<Real>(sc, y.data(), grad, e, gy.data());
      store(i, y.data(), e, gy.data());
      nr[i] = e.nrays; nf[i] = e.nonfinite; accepted[i] = 1;
    }
    for (uint32_t i = 0; i < N; ++i) { rays += nr[i]; nonfinite += nf[i]; }
    bootstrap();
    for (uint32_t i = 0; i < N; ++i) accumulate(i, 0);
    rebuild_queue();
  }

  void rebuild_queue() {
    queue.clear();
    for (uint32_t i = 0; i < N; ++i) if (killed[i]) queue.push_back(i);
  }

  // ln q(a -> b) of the MALA proposal, minimal-image difference (Q11)
  Real log_q(const Real* a, const Real* ga, const Real* b) const {
    const Real s = (Real)cfg.stddev, h = Real(0.5) * s * s;
    Real acc = 0;
    for (uint32_t j = 0; j < d; ++j) {
      const Real dl = min_image<Real>(b[j] - a[j] - h * ga[j]);
      acc += dl * dl;
    }
    return -acc / (Real(2) * s * s);
  }

  // Alg. 2 for every chain, `iters` times.
  void step(uint32_t iters) {
    const Real s = (Real)cfg.stddev, h = Real(0.5) * s * s, ct = (Real)cfg.c_tilde;
    std::vector<Real> Y((size_t)N * d), GY((size_t)N * d);
    std::vector<Eval<Real>> E(N);
    std::vector<uint8_t> kind(N);  // 0 local, 1 regeneration, 2 large step
    for (uint32_t it = 0; it < iters; ++it) {
      const uint32_t n = ++iteration;
      kills_last = 0;
#pragma omp parallel for schedule(dynamic, 64)
      for (int64_t ii = 0; ii < (int64_t)N; ++ii) {
        const uint32_t i = (uint32_t)ii;
        Real* y = &Y[(size_t)i * d];
        const Real* xi_ = &x[(size_t)i * d];
        const Real* gi = &g[(size_t)i * d];
        uint32_t w[4];
        stream_block(cfg.seed, cfg.chain_offset + i, n, 0, DECIDE, epoch, w);
        if ((restore && killed[i]) || cfg.method == PATH_TRACING) {   // Alg. 2: re-initialise from nu; PT: always
          kind[i] = 1;
          uniform_point(i, n, REGEN_U, y);
          if (restore) regeneration_point(y);
        } else if (!restore && u01_co<Real>(w[0]) < (Real)cfg.large_step_prob) {
          kind[i] = 2;                              // large step (plain MH only), L747
          uniform_point(i, n, LARGE_U, y);
        } else {                                    // LocalDynamics
          kind[i] = 0;
          std::vector<Real> xi(d);
          normals(i, n, xi.data());
          if (cfg.method == DIFFUSION_RESTORE && cfg.a_mode == 1) {   // another antisymmetric pattern (Q24): x_j += c~ (A~ g)_j
            for (uint32_t b = 0; b < d; b += 4) {
              const bool four = b + 3 < d;                             // a trailing 2-block keeps the paper's rotation
              const uint32_t p0 = four ? b + 2 : b + 1, p1 = four ? b + 3 : b;
              Real r[4] = {ct * gi[p0], four ? ct * gi[p1] : -(ct * gi[p1]), Real(0), Real(0)};
              if (four) { r[2] = -(ct * gi[b]); r[3] = -(ct * gi[b + 1]); }
              for (uint32_t c = 0; c < (four ? 4u : 2u); ++c)
                y[b + c] = wrap01<Real>(((xi_[b + c] + h * gi[b + c]) + r[c]) + s * xi[b + c]);
            }
          } else if (cfg.method == DIFFUSION_RESTORE) {    // Alg. 4
            for (uint32_t b = 0; b < d; b += 2) {
              const Real r0 = ct * gi[b + 1], r1 = -(ct * gi[b]);     // rotate(v) = c~ (v2, -v1), L720
              y[b] = wrap01<Real>(((xi_[b] + h * gi[b]) + r0) + s * xi[b]);
              y[b + 1] = wrap01<Real>(((xi_[b + 1] + h * gi[b + 1]) + r1) + s * xi[b + 1]);
            }
          } else if (grad) {                        // MALA proposal
            for (uint32_t j = 0; j < d; ++j) y[j] = wrap01<Real>((xi_[j] + h * gi[j]) + s * xi[j]);
          } else {                                  // Metropolis proposal
            for (uint32_t j = 0; j < d; ++j) y[j] = wrap01<Real>(xi_[j] + s * xi[j]);
          }
        }
        evaluate<Real>(sc, y, grad, E[i], &GY[(size_t)i * d]);
      }
      for (uint32_t i = 0; i < N; ++i) {
        uint32_t w[4];
        stream_block(cfg.seed, cfg.chain_offset + i, n, 0, DECIDE, epoch, w);
        const Real* y = &Y[(size_t)i * d];
        const Real* gy = &GY[(size_t)i * d];
        rays += E[i].nrays; nonfinite += E[i].nonfinite;
        bool take = true;
        if (kind[i] != 1 && cfg.method != DIFFUSION_RESTORE) {   // Metropolis-Hastings test
          const Real px = p[i] + Real(kEps), py = E[i].p + Real(kEps);
          Real a = py / px;
          if (kind[i] == 0 && grad)
            a *= std::exp(log_q(y, gy, &x[(size_t)i * d]) - log_q(&x[(size_t)i * d], &g[(size_t)i * d], y));
          if (!(a < Real(1))) a = Real(1);
          take = u01_co<Real>(w[1]) < a;
          if (take) ++mh_accepts;
        }
        accepted[i] = take;
        if (take) store(i, y, E[i], gy);
        accumulate(i, n);                                        // Alg. 2
      }
      rebuild_queue();
    }
  }

  // Alg. 3 (L548) with the pixel-count factor of Q2; plain MH: p_lambda / N_mut (Q11).
  // Returns 1 (warning) and a zero image when no tour has completed yet.
  int resolve(double* rgb) const {
    double scale;
    if (restore) {
      if (tours == 0) { std::fill(rgb, rgb + (size_t)npix * 3, 0.0); return 1; }
      scale = (double)npix * (double)kappa0 / (double)tours;
    } else if (cfg.method == PATH_TRACING) {
      scale = (double)npix / (double)mutations;                 // mean of f over the samples, per pixel area
    } else {
      scale = (double)npix * (double)p_lambda / (double)mutations;
    }
    for (uint32_t q = 0; q < npix; ++q)
      for (int c = 0; c < 3; ++c) rgb[(size_t)q * 3 + c] = scale * accum[(size_t)q * 4 + c];
    return 0;
  }
};

// Ordinary path tracing: independent uniform PSS samples, the reference the
// MCMC estimators must agree with at convergence.  image[pix] += f * N_pix / n.
template <class Real> void pt_render(const Scene<Real>& sc, uint64_t n, uint64_t seed, double* rgb) {
  const uint32_t d = sc.dim(), npix = sc.W * sc.H;
  std::fill(rgb, rgb + (size_t)npix * 3, 0.0);
  const uint64_t chunk = 1u << 16;
  std::vector<Eval<Real>> E(chunk);
  for (uint64_t base = 0; base < n; base += chunk) {
    const uint64_t cnt = std::min(chunk, n - base);
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t k = 0; k < (int64_t)cnt; ++k) {
      const uint64_t i = base + (uint64_t)k;
      std::vector<Real> y(d);
      for (uint32_t j = 0; j < d; j += 4) {
        uint32_t w[4];
        stream_block(seed, (uint32_t)i, (uint32_t)(i >> 32), j / 4, REGEN_U, 0xFFFFFFu, w);
        for (uint32_t c = 0; c < 4 && j + c < d; ++c) y[j + c] = u01_co<Real>(w[c]);
      }
      evaluate<Real>(sc, y.data(), false, E[k], nullptr);
    }
    const double wgt = (double)npix / (double)n;
    for (uint64_t k = 0; k < cnt; ++k)
      for (int c = 0; c < 3; ++c) rgb[(size_t)E[k].pix * 3 + c] += wgt * (double)E[k].f[c];
  }
}

}  // namespace orc
