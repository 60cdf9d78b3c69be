// TEST INFRASTRUCTURE — CPU oracle (see philox.hpp header).
//
// Plain C entry points over the templated oracle so that tests/ and bench.py's
// cpu_baseline leg can drive it through ctypes (oracle/oracle.py).  All floating-point
// data crosses this boundary as double; `prec` = 0 runs the oracle in float (the
// precision the kernels decide in — used for parity), 1 in double (used for the pins).
#include <omp.h>

#include <cstdint>
#include <cstring>
#include <memory>
#include <vector>

#include "bias.hpp"
#include "samplers.hpp"

using namespace orc;

namespace {

struct SceneH {
  int prec;
  Scene<float> f;
  Scene<double> d;
};
struct ChainsH {
  int prec;
  std::unique_ptr<Chains<float>> f;
  std::unique_ptr<Chains<double>> d;
};

template <class Real>
void fill_scene(Scene<Real>& sc, const float* verts, uint32_t nv, const uint32_t* idx, uint32_t nt, const uint32_t* tri_mat,
                const double* mats, uint32_t nm, const float* env, const float* cam, float vfov, uint32_t W, uint32_t H,
                uint32_t L, int use_bvh, int nee) {
  sc.set_geometry(verts, nv, idx, nt);
  sc.tri_mat.assign(tri_mat, tri_mat + nt);
  sc.mats.resize(nm);
  for (uint32_t i = 0; i < nm; ++i) {
    const double* m = mats + 9 * i;  // kind, a0,a1,a2, ior, alpha, Le0,Le1,Le2 (values are float32-exact)
    sc.mats[i].kind = (int)m[0];
    for (int c = 0; c < 3; ++c) { sc.mats[i].a[c] = (Real)m[1 + c]; sc.mats[i].Le[c] = (Real)m[6 + c]; }
    sc.mats[i].ior = (Real)m[4]; sc.mats[i].alpha = (Real)m[5];
  }
  for (int c = 0; c < 3; ++c) sc.env[c] = (Real)env[c];
  sc.set_camera(cam, cam + 3, cam + 6, vfov, W, H);
  sc.L = L; sc.use_bvh = use_bvh != 0;
  sc.nee = nee != 0;
  sc.build_lights();
}

template <class Real>
void fill_analytic(Scene<Real>& sc, uint32_t nc, const double* w, const double* mx, const double* my, const double* s, uint32_t W, uint32_t H) {
  sc.analytic = true; sc.W = W; sc.H = H; sc.L = 1;
  for (uint32_t k = 0; k < nc; ++k) {
    sc.mix_w.push_back((Real)w[k]); sc.mix_mx.push_back((Real)mx[k]);
    sc.mix_my.push_back((Real)my[k]); sc.mix_s.push_back((Real)s[k]);
  }
}

template <class Real>
void do_trace(const Scene<Real>& sc, const double* o, const double* d, uint32_t n, int mode, double* t, int32_t* tri) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    const Vec3<Real> ov{(Real)o[3 * i], (Real)o[3 * i + 1], (Real)o[3 * i + 2]};
    const Vec3<Real> dv{(Real)d[3 * i], (Real)d[3 * i + 1], (Real)d[3 * i + 2]};
    const Hit<Real> h = mode == 0 ? sc.intersect_brute(ov, dv) : sc.intersect_bvh(ov, dv);
    t[i] = h.ok ? (double)h.t : -1.0;
    tri[i] = h.ok ? (int32_t)h.tri : -1;
  }
}

template <class Real>
void do_eval(const Scene<Real>& sc, const double* x, uint32_t n, int want_score, double* f, double* p, uint32_t* pix,
             uint32_t* nrays, uint32_t* sig, double* g, uint8_t* nonfinite) {
  const uint32_t d = sc.dim();
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < (int64_t)n; ++i) {
    std::vector<Real> xs(d), gs(d);
    for (uint32_t j = 0; j < d; ++j) xs[j] = (Real)x[(size_t)i * d + j];
    Eval<Real> e;
    evaluate<Real>(sc, xs.data(), want_score != 0, e, gs.data());
    for (int c = 0; c < 3; ++c) f[3 * i + c] = (double)e.f[c];
    p[i] = (double)e.p; pix[i] = e.pix; nrays[i] = e.nrays; sig[i] = e.sig; nonfinite[i] = e.nonfinite;
    if (want_score) for (uint32_t j = 0; j < d; ++j) g[(size_t)i * d + j] = (double)gs[j];
  }
}

template <class Real>
void get_state(const Chains<Real>& c, double* x, double* p, double* fop, uint32_t* pix, uint8_t* killed, double* g, uint32_t* sig) {
  for (size_t k = 0; k < c.x.size(); ++k) { x[k] = (double)c.x[k]; g[k] = (double)c.g[k]; }
  for (uint32_t i = 0; i < c.N; ++i) { p[i] = (double)c.p[i]; pix[i] = c.pix[i]; killed[i] = c.killed[i]; sig[i] = c.sig[i]; }
  for (size_t k = 0; k < c.fop.size(); ++k) fop[k] = (double)c.fop[k];
}
template <class Real>
void set_state(Chains<Real>& c, const double* x, const double* p, const double* fop, const uint32_t* pix, const uint8_t* killed,
               const double* g, uint32_t iteration) {
  for (size_t k = 0; k < c.x.size(); ++k) { c.x[k] = (Real)x[k]; c.g[k] = (Real)g[k]; }
  for (uint32_t i = 0; i < c.N; ++i) { c.p[i] = (Real)p[i]; c.pix[i] = pix[i]; c.killed[i] = killed[i]; }
  for (size_t k = 0; k < c.fop.size(); ++k) c.fop[k] = (Real)fop[k];
  c.iteration = iteration;
  c.rebuild_queue();
}

#define WITH_SCENE(h, S, body) do { if ((h)->prec == 0) { auto& S = (h)->f; body; } else { auto& S = (h)->d; body; } } while (0)
#define WITH_CHAINS(h, C, body) do { if ((h)->prec == 0) { auto& C = *(h)->f; body; } else { auto& C = *(h)->d; body; } } while (0)

}  // namespace

extern "C" {

void orc_set_threads(int n) { omp_set_num_threads(n); }
int orc_max_threads() { return omp_get_max_threads(); }

void orc_philox(const uint32_t* key, const uint32_t* ctr, uint32_t* out) { philox4x32_10(key, ctr, out); }
void orc_stream_block(uint64_t seed, uint32_t chain, uint32_t iter, uint32_t slot, uint32_t purpose, uint32_t epoch, uint32_t* out) {
  stream_block(seed, chain, iter, slot, purpose, epoch, out);
}
// out[0] = u in [0,1), out[1] = u in (0,1], out[2..3] = Box-Muller pair from (w, w2)
void orc_rng_transforms(uint32_t w, uint32_t w2, int prec, double* out) {
  if (prec == 0) {
    float a, b; box_muller<float>(w, w2, a, b);
    out[0] = u01_co<float>(w); out[1] = u01_oc<float>(w); out[2] = a; out[3] = b;
  } else {
    double a, b; box_muller<double>(w, w2, a, b);
    out[0] = u01_co<double>(w); out[1] = u01_oc<double>(w); out[2] = a; out[3] = b;
  }
}
double orc_wrap(double v, int prec) { return prec == 0 ? (double)wrap01<float>((float)v) : wrap01<double>(v); }
double orc_min_image(double v, int prec) { return prec == 0 ? (double)min_image<float>((float)v) : min_image<double>(v); }

void* orc_scene_create(int prec, const float* verts, uint32_t nv, const uint32_t* idx, uint32_t nt, const uint32_t* tri_mat,
                       const double* mats, uint32_t nm, const float* env, const float* cam, float vfov, uint32_t W, uint32_t H,
                       uint32_t L, int use_bvh, int nee) {
  auto* h = new SceneH();
  h->prec = prec;
  WITH_SCENE(h, S, fill_scene(S, verts, nv, idx, nt, tri_mat, mats, nm, env, cam, vfov, W, H, L, use_bvh, nee));
  return h;
}
void* orc_scene_create_analytic2d(int prec, uint32_t nc, const double* w, const double* mx, const double* my, const double* s, uint32_t W, uint32_t H) {
  auto* h = new SceneH();
  h->prec = prec;
  WITH_SCENE(h, S, fill_analytic(S, nc, w, mx, my, s, W, H));
  return h;
}
void orc_scene_destroy(void* h) { delete (SceneH*)h; }
uint32_t orc_scene_dim(void* h_) { auto* h = (SceneH*)h_; uint32_t r = 0; WITH_SCENE(h, S, r = S.dim()); return r; }
double orc_scene_eps_ray(void* h_) { auto* h = (SceneH*)h_; double r = 0; WITH_SCENE(h, S, r = (double)S.eps_ray); return r; }

void orc_trace(void* h_, const double* o, const double* d, uint32_t n, int mode, double* t, int32_t* tri) {
  auto* h = (SceneH*)h_;
  WITH_SCENE(h, S, do_trace(S, o, d, n, mode, t, tri));
}
void orc_eval(void* h_, const double* x, uint32_t n, int want_score, double* f, double* p, uint32_t* pix, uint32_t* nrays,
              uint32_t* sig, double* g, uint8_t* nonfinite) {
  auto* h = (SceneH*)h_;
  WITH_SCENE(h, S, do_eval(S, x, n, want_score, f, p, pix, nrays, sig, g, nonfinite));
}
void orc_pt_render(void* h_, uint64_t n, uint64_t seed, double* rgb) {
  auto* h = (SceneH*)h_;
  WITH_SCENE(h, S, pt_render(S, n, seed, rgb));
}

// Appendix-C bias field of the analytic target on a G x G grid (bias.hpp); M x M quadrature points
void orc_bias_field(void* h_, double stddev, double c_tilde, double dt, uint32_t G, uint32_t M, double* out) {
  auto* h = (SceneH*)h_;
  if (h->prec == 0) bias_field<float>(h->f, (float)stddev, (float)c_tilde, (float)dt, G, M, out);
  else bias_field<double>(h->d, stddev, c_tilde, dt, G, M, out);
}

void* orc_chains_create(void* scene_, int method, uint32_t n_chains, double stddev, double c_tilde, double dt, double m,
                        double large_step_prob, double p_lambda_override, uint64_t seed, uint32_t chain_offset, int rao_blackwell) {
  auto* s = (SceneH*)scene_;
  auto* h = new ChainsH();
  h->prec = s->prec;
  Config c{method, n_chains, stddev, c_tilde, dt, m, large_step_prob, p_lambda_override, seed, chain_offset, rao_blackwell};
  if (s->prec == 0) h->f.reset(new Chains<float>(s->f, c)); else h->d.reset(new Chains<double>(s->d, c));
  return h;
}
void orc_chains_destroy(void* h) { delete (ChainsH*)h; }
// f4 (Q24): a_mode and the regeneration density (G x G tile probabilities summing to one; G = 0: uniform); before init
void orc_chains_set_f4(void* h_, int a_mode, uint32_t G, const double* w) {
  auto* h = (ChainsH*)h_;
  WITH_CHAINS(h, C, { C.cfg.a_mode = a_mode; C.cfg.rho_grid = G; C.cfg.rho_w.assign(w, w + (size_t)G * G); });
}
void orc_chains_init(void* h_, uint32_t frame) { auto* h = (ChainsH*)h_; WITH_CHAINS(h, C, C.init(frame)); }
void orc_chains_step(void* h_, uint32_t iters) { auto* h = (ChainsH*)h_; WITH_CHAINS(h, C, C.step(iters)); }
void orc_chains_get_state(void* h_, double* x, double* p, double* fop, uint32_t* pix, uint8_t* killed, double* g, uint32_t* sig) {
  auto* h = (ChainsH*)h_; WITH_CHAINS(h, C, get_state(C, x, p, fop, pix, killed, g, sig));
}
void orc_chains_set_state(void* h_, const double* x, const double* p, const double* fop, const uint32_t* pix, const uint8_t* killed,
                          const double* g, uint32_t iteration) {
  auto* h = (ChainsH*)h_; WITH_CHAINS(h, C, set_state(C, x, p, fop, pix, killed, g, iteration));
}
// accepted flag and sampled weight (dtau, or 1 for plain MH) of every chain's last step
void orc_chains_last(void* h_, uint8_t* accepted, double* dtau) {
  auto* h = (ChainsH*)h_;
  WITH_CHAINS(h, C, { for (uint32_t i = 0; i < C.N; ++i) { accepted[i] = C.accepted[i]; dtau[i] = (double)C.dtau[i]; } });
}
void orc_chains_accum(void* h_, double* out) { auto* h = (ChainsH*)h_; WITH_CHAINS(h, C, std::memcpy(out, C.accum.data(), C.accum.size() * sizeof(double))); }
void orc_chains_zero_accum(void* h_) { auto* h = (ChainsH*)h_; WITH_CHAINS(h, C, std::fill(C.accum.begin(), C.accum.end(), 0.0)); }
int orc_chains_resolve(void* h_, double* rgb) { auto* h = (ChainsH*)h_; int r = 0; WITH_CHAINS(h, C, r = C.resolve(rgb)); return r; }
// out: tours, mutations, rays, mh_accepts, nonfinite, kills_last, queue_len, p_lambda, kappa0, lambda, iteration
void orc_chains_stats(void* h_, double* out) {
  auto* h = (ChainsH*)h_;
  WITH_CHAINS(h, C, {
    out[0] = (double)C.tours; out[1] = (double)C.mutations; out[2] = (double)C.rays; out[3] = (double)C.mh_accepts;
    out[4] = (double)C.nonfinite; out[5] = (double)C.kills_last; out[6] = (double)C.queue.size();
    out[7] = (double)C.p_lambda; out[8] = (double)C.kappa0; out[9] = (double)C.lambda; out[10] = (double)C.iteration;
  });
}
uint32_t orc_chains_queue(void* h_, uint32_t* ids) {
  auto* h = (ChainsH*)h_; uint32_t n = 0;
  WITH_CHAINS(h, C, { n = (uint32_t)C.queue.size(); if (ids) std::memcpy(ids, C.queue.data(), n * sizeof(uint32_t)); });
  return n;
}

}  // extern "C"
