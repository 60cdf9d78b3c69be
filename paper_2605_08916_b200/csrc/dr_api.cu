// C-ABI entry points (include/dr.h): argument validation, scene upload, state layout, kernel launches.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/dr.h"
#include "dr_kernels.cuh"
#include "dr_wave.cuh"
#include "dr_grad.cuh"

using namespace dr;

namespace {

thread_local std::string g_err;

dr_status fail(dr_status s, const std::string& msg) { g_err = msg; return s; }

#define CUDA_TRY(expr)                                                                                   \
  do {                                                                                                   \
    cudaError_t e_ = (expr);                                                                             \
    if (e_ != cudaSuccess)                                                                               \
      return fail(e_ == cudaErrorMemoryAllocation ? DR_ERR_OOM : DR_ERR_CUDA,                            \
                  std::string(#expr) + ": " + cudaGetErrorString(e_));                                   \
  } while (0)

size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

constexpr uint32_t kWaveMaxStates = 1u << 21;   // very large evaluations use the per-segment loop: their launches are long enough for the tail
                                                // not to matter, and k_trace's 20 trace warps beat k_wave's 17 (profiles/r01g_sweep.md vs r01f_sweep.md)
constexpr size_t kMaxDynSmem = 227 * 1024;  // opt-in shared memory per block on sm_100

bool finite3(const float* v) { return std::isfinite(v[0]) && std::isfinite(v[1]) && std::isfinite(v[2]); }

void normalize(float* v) {   // a * (1 / |a|), the form used everywhere (dr_path.cuh)
  const float inv = 1.0f / std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
  v[0] *= inv; v[1] *= inv; v[2] *= inv;
}
void cross(const float* a, const float* b, float* c) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

}  // namespace

struct dr_scene {
  DevScene dev{};
  void* d_nodes = nullptr;
  void* d_tris = nullptr;
  void* d_mats = nullptr;
  void* d_lights = nullptr;
  dr_scene_info info{};
  int n_sm = 1;            // persistent k_trace grid: one block per SM
  size_t trace_smem = 0;   // per-thread traversal stacks
  bool wave_ok = false;    // k_wave's shared memory (trace_smem + kWaveExtraSmem) fits; otherwise every evaluation uses the loop
};

struct dr_chains {
  const dr_scene* scene = nullptr;
  dr_config cfg{};
  ChainParams cp{};
  ChainState st{};
  float4* accum = nullptr;
  uint32_t npix = 0, nblocks = 0;
  uint32_t iteration = 0;
  bool initialised = false;
  size_t state_bytes = 0;
  void* state_base = nullptr;
  // optional per-kernel timing (dr_profile_*): cudaEvent pairs recorded around every launch
  bool profiling = false;
  std::vector<cudaEvent_t> ev;     // pool
  std::vector<int> ev_kind;        // kernel class of pair k (events 2k, 2k+1)
  size_t ev_used = 0;              // pairs in use
  double prof_ms[DR_PROF_COUNT] = {};
  uint64_t prof_launches[DR_PROF_COUNT] = {};
  EvalWs ws{};
  uint32_t eval_tag = 0;           // k_wave: tag of the last evaluation (dr_wave.cuh)
  int eval_form = 0;               // test hook dr_chains_set_eval_form: 0 = default choice, 1 = per-segment loop, 2 = k_wave, 3 / 4 = k_wave in the small / big block shape
  void* hook_scratch = nullptr;    // device staging of dr_chains_download / _upload (row-major copies), allocated on first use
  void* d_rho = nullptr;           // f4: (probability, running sum) per film tile
  uint32_t* h_last_rays = nullptr; // pinned: rays of the last k_wave evaluation that has finished (copied behind every evaluation, read
                                   // without waiting: it picks the block shape of the next one, which does not change any result)
  ~dr_chains() { for (cudaEvent_t e : ev) cudaEventDestroy(e); cudaFree(hook_scratch); cudaFree(d_rho); if (h_last_rays) cudaFreeHost(h_last_rays); }
};

namespace {

struct Layout {
  size_t x, g, fp, pix, sig, killed, y, gy, fy, pixy, sigy, kind, accepted, weight, order, blockcnt, blockoff, partial, ctr;
  size_t q, hits, ring, rec, vrec, adj, pinfo, gradlist, ctl;   // evaluation workspace (dr_eval.cuh EvalWs)
  size_t total;
};

Layout make_layout(uint32_t N, uint32_t planes, uint32_t Lseg, bool grad, bool nee) {
  Layout L{};
  size_t o = 0;
  auto take = [&](size_t bytes) { const size_t at = o; o = align256(o + bytes); return at; };
  const size_t nb = (N + kBlock - 1) / kBlock;
  L.x = take(sizeof(float4) * planes * N);
  L.g = take(grad ? sizeof(float4) * planes * N : 0);
  L.fp = take(sizeof(float4) * N);
  L.pix = take(4 * (size_t)N);
  L.sig = take(4 * (size_t)N);
  L.killed = take(N);
  L.y = take(sizeof(float4) * planes * N);
  L.gy = take(grad ? sizeof(float4) * planes * N : 0);
  L.fy = take(sizeof(float4) * N);
  L.pixy = take(4 * (size_t)N);
  L.sigy = take(4 * (size_t)N);
  L.kind = take(N);
  L.accepted = take(N);
  L.weight = take(4 * (size_t)N);
  L.order = take(4 * (size_t)N);
  L.blockcnt = take(4 * nb);
  L.blockoff = take(4 * nb);
  L.partial = take(8 * nb);
  L.ctr = take(sizeof(Counters));
  L.q = take(6 * sizeof(float4) * (size_t)N);           // qa | qb, or the 64-byte ray records of k_wave
  L.hits = take(sizeof(uint2) * (size_t)N);
  L.ring = take(sizeof(uint2) * (size_t)N * (nee ? 2 * Lseg - 1 : Lseg));   // one entry per ray of an evaluation, never reused (dr_wave.cuh)
  L.rec = take(grad ? sizeof(float4) * (size_t)N * (nee ? 1 : Lseg) : 0);
  L.vrec = take(grad && nee ? 3 * sizeof(float4) * (size_t)N * Lseg : 0);
  L.adj = take(grad && nee ? sizeof(float4) * (size_t)N * 3 : 0);
  L.pinfo = take(grad ? 4 * (size_t)N : 0);
  L.gradlist = take(grad ? 4 * (size_t)N * (nee ? 3 * Lseg : 1) : 0);   // with next-event estimation: one list per (vertex index, material kind)
  L.ctl = take(4 * kCtlWords);
  L.total = o;
  return L;
}

dr_status check_config(const dr_config* c) {
  if (!c) return fail(DR_ERR_INVALID_ARG, "config is null");
  if (c->method < 0 || c->method > DR_PATH_TRACING) return fail(DR_ERR_INVALID_ARG, "method out of range");
  if (c->rao_blackwell > 1) return fail(DR_ERR_INVALID_ARG, "rao_blackwell must be 0 or 1");
  if (c->a_mode > 1) return fail(DR_ERR_INVALID_ARG, "a_mode must be 0 or 1");
  if (c->rho_grid > 64) return fail(DR_ERR_INVALID_ARG, "rho_grid must be <= 64");
  if (c->rho_grid && c->method == DR_PATH_TRACING)   // its samples are averaged with unit weight: a non-uniform first draw would bias the image
    return fail(DR_ERR_INVALID_ARG, "rho_grid must be 0 for DR_PATH_TRACING (path tracing draws every sample uniformly)");
  if (c->rho_grid) {
    if (!c->host_rho) return fail(DR_ERR_INVALID_ARG, "rho_grid > 0 needs host_rho");
    double sum = 0.0;
    for (uint32_t t = 0; t < c->rho_grid * c->rho_grid; ++t) {
      if (!std::isfinite(c->host_rho[t])) return fail(DR_ERR_NONFINITE, "non-finite tile probability");
      if (!(c->host_rho[t] > 0.f)) return fail(DR_ERR_INVALID_ARG, "tile probabilities must be > 0");
      sum += c->host_rho[t];
    }
    if (std::fabs(sum - 1.0) > 1e-4) return fail(DR_ERR_INVALID_ARG, "tile probabilities must sum to one");
  }
  if (c->n_chains < 1) return fail(DR_ERR_INVALID_ARG, "n_chains must be >= 1");
  if (!(c->stddev > 0.f) || !std::isfinite(c->stddev)) return fail(DR_ERR_INVALID_ARG, "stddev must be > 0");
  if (!(c->c_tilde >= 0.f) || !std::isfinite(c->c_tilde)) return fail(DR_ERR_INVALID_ARG, "c_tilde must be >= 0");
  if (!(c->dt > 0.f) || !std::isfinite(c->dt)) return fail(DR_ERR_INVALID_ARG, "dt must be > 0");
  if (!(c->m > 0.f) || !std::isfinite(c->m)) return fail(DR_ERR_INVALID_ARG, "m must be > 0");
  if (!(c->large_step_prob >= 0.f && c->large_step_prob <= 1.f)) return fail(DR_ERR_INVALID_ARG, "large_step_prob must be in [0,1]");
  if (!std::isfinite(c->p_lambda_override)) return fail(DR_ERR_INVALID_ARG, "p_lambda_override must be finite");
  return DR_OK;
}

constexpr size_t kMaxPairs = 8192;

// Folds finished event pairs into the per-class totals (requires the stream to be idle).
void prof_drain(dr_chains* c) {
  for (size_t k = 0; k < c->ev_used; ++k) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->ev[2 * k], c->ev[2 * k + 1]) == cudaSuccess) {
      c->prof_ms[c->ev_kind[k] & 0xFF] += ms;
      c->prof_launches[c->ev_kind[k] & 0xFF] += (uint64_t)(c->ev_kind[k] >> 8);   // kernel launches inside the pair
    }
  }
  c->ev_used = 0;
}

struct ProfScope {
  dr_chains* c; cudaStream_t s; size_t k; bool on;
  ProfScope(dr_chains* c_, int kind, cudaStream_t s_, int launches = 1) : c(c_), s(s_), k(0), on(c_ && c_->profiling) {
    if (!on) return;
    if (c->ev_used == kMaxPairs) { cudaStreamSynchronize(s); prof_drain(c); }
    k = c->ev_used++;
    while (c->ev.size() < 2 * (k + 1)) { cudaEvent_t e; cudaEventCreate(&e); c->ev.push_back(e); }
    if (c->ev_kind.size() <= k) c->ev_kind.resize(k + 1);
    c->ev_kind[k] = kind | (launches << 8);
    cudaEventRecord(c->ev[2 * k], s);
  }
  ~ProfScope() { if (on) cudaEventRecord(c->ev[2 * k + 1], s); }
};

// Rows a3-a6 for n states (dr_eval.cuh): raygen, then trace + shade of every segment, then the reverse pass.
// prof may be null (test hooks).  io.g must be zero on entry when grad is set.  form: 0 = default (one persistent
// k_wave launch, in the small block shape below kWaveSmallBelow states; the per-segment loop for the counting pass and for very
// large n), 1 = loop, 2 = k_wave, 3 / 4 = k_wave in the small / big block shape.
// shared memory of a traversal block of `block` threads: one constant word + per-thread node and triangle stacks
size_t trace_stack_bytes(uint32_t stack_cap, int block) {
  return ((size_t)(stack_cap + kTriStack) * sizeof(uint2) + (size_t)kTriStack * sizeof(uint32_t)) * block + 16;
}

// k_wave in the block shape C (dr_eval.cuh TraceBig / TraceSmall)
template <class C>
void launch_wave(const DevScene& dev, const EvalWs& ws, const EvalIO& io, uint32_t n, bool grad, bool stats, int n_sm, cudaStream_t s) {
  const size_t sm = trace_stack_bytes(dev.stack_cap, C::kBlock) + kWaveExtraSmem;
  if (dev.nee) {
    if (stats) {   // the counting pass of a scene with next-event estimation (others count in k_trace<true>)
      if (grad) k_wave<true, true, true, C><<<n_sm, C::kBlock, sm, s>>>(dev, ws, io, n);
      else k_wave<false, true, true, C><<<n_sm, C::kBlock, sm, s>>>(dev, ws, io, n);
    } else if (grad) k_wave<true, false, true, C><<<n_sm, C::kBlock, sm, s>>>(dev, ws, io, n);
    else k_wave<false, false, true, C><<<n_sm, C::kBlock, sm, s>>>(dev, ws, io, n);
  } else if (grad) k_wave<true, false, false, C><<<n_sm, C::kBlock, sm, s>>>(dev, ws, io, n);
  else k_wave<false, false, false, C><<<n_sm, C::kBlock, sm, s>>>(dev, ws, io, n);
}
template <class C>
cudaError_t wave_allow_smem() {
  const void* waves[] = {(const void*)k_wave<false, false, false, C>, (const void*)k_wave<true, false, false, C>, (const void*)k_wave<false, false, true, C>,
                         (const void*)k_wave<true, false, true, C>, (const void*)k_wave<false, true, true, C>, (const void*)k_wave<true, true, true, C>};
  cudaError_t e = cudaSuccess;
  for (const void* w : waves)
    if (e == cudaSuccess) e = cudaFuncSetAttribute(w, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem);
  return e;
}

dr_status launch_eval(dr_chains* prof, const dr_scene* sc, EvalWs ws, const EvalIO& io, uint32_t n, bool grad, bool stats,
                      int form, cudaStream_t s) {
  const DevScene& dev = sc->dev;
  const uint32_t g = (n + kShadeBlock - 1) / kShadeBlock;
  if (dev.analytic) {
    ProfScope ps(prof, DR_PROF_SHADE, s);
    if (grad) k_eval_analytic<true><<<g, kShadeBlock, 0, s>>>(dev, io, n);
    else k_eval_analytic<false><<<g, kShadeBlock, 0, s>>>(dev, io, n);
    CUDA_TRY(cudaGetLastError());
    return DR_OK;
  }
  if (form < 0 || form > 4) return fail(DR_ERR_INVALID_ARG, "evaluation form must be 0 .. 4");
  if (dev.nee && (!sc->wave_ok || form == 1)) return fail(DR_ERR_UNSUPPORTED, "next-event estimation runs in k_wave only (no per-segment loop)");
  const bool wave = dev.nee || (!stats && sc->wave_ok && (form >= 2 || (form == 0 && n < kWaveMaxStates)));
  if (wave && n > kWaveStateMask) return fail(DR_ERR_UNSUPPORTED, "k_wave addresses at most 2^27 states per evaluation");
  CUDA_TRY(cudaMemsetAsync(ws.ctl, 0, 4 * kCtlWords, s));
  {
    ProfScope ps(prof, DR_PROF_RAYGEN, s);
    if (wave) k_raygen<true><<<g, kShadeBlock, 0, s>>>(dev, ws, io, n);
    else k_raygen<false><<<g, kShadeBlock, 0, s>>>(dev, ws, io, n);
  }
#if DR_CHECKS
  if (wave) CUDA_TRY(cudaMemsetAsync(ws.hits, 0, sizeof(uint2) * (size_t)ws.cap, s));   // per-state segment counters of the checks
#endif
  if (wave) {
    ProfScope ps(prof, DR_PROF_TRACE, s);
    // the block shape: by the rays the ensemble's last finished evaluation made, if that is known, else by the number of states
    bool small = n < (dev.nee ? kWaveSmallBelowNee : kWaveSmallBelow);
    const uint32_t last_rays = prof && prof->h_last_rays ? *(volatile uint32_t*)prof->h_last_rays : 0u;
    if (last_rays) small = last_rays < kWaveSmallBelowRays;
    if (form == 3) small = true;
    if (form == 4) small = false;
    if (small) launch_wave<TraceSmall>(dev, ws, io, n, grad, stats, sc->n_sm, s);
    else launch_wave<TraceBig>(dev, ws, io, n, grad, stats, sc->n_sm, s);
    if (prof && prof->h_last_rays && !stats) cudaMemcpyAsync(prof->h_last_rays, ws.ctl + kCtlWaveReserve, 4, cudaMemcpyDeviceToHost, s);
  } else
  for (uint32_t k = 1; k <= dev.L; ++k) {
    const float4* q = (k & 1u) ? ws.qa : ws.qb;
    {
      ProfScope ps(prof, DR_PROF_TRACE, s);
      if (stats) k_trace<true><<<sc->n_sm, kTraceBlock, sc->trace_smem, s>>>(dev, q, ws.cap, ws.ctl + kCtlCnt + k, ws.ctl + kCtlHead + k, ws.hits, io.work);
      else k_trace<false><<<sc->n_sm, kTraceBlock, sc->trace_smem, s>>>(dev, q, ws.cap, ws.ctl + kCtlCnt + k, ws.ctl + kCtlHead + k, ws.hits, io.work);
    }
    {
      ProfScope ps(prof, DR_PROF_SHADE, s);
      if (grad) k_shade<true><<<g, kShadeBlock, 0, s>>>(dev, ws, io, k);
      else k_shade<false><<<g, kShadeBlock, 0, s>>>(dev, ws, io, k);
    }
  }
  if (grad) {
    ProfScope ps(prof, DR_PROF_GRAD, s, dev.nee ? (int)dev.L + 1 : 1);   // with next-event estimation: init, L - 1 vertex launches, finish
    if (dev.nee) {   // one launch per vertex index and material kind, last vertex first (dr_grad.cuh)
      k_grad_nee_init<<<(n + kGradInitBlock - 1) / kGradInitBlock, kGradInitBlock, 0, s>>>(dev, ws, io, n);
      const uint32_t gv = (n + kGradVertexBlock - 1) / kGradVertexBlock + 3;   // three lists, each rounded up to whole blocks
      for (uint32_t k = dev.L - 1; k >= 1; --k) k_grad_nee_vertex<<<gv, kGradVertexBlock, 0, s>>>(dev, ws, io, k);
      k_grad_nee_finish<<<(n + kGradBlock - 1) / kGradBlock, kGradBlock, 0, s>>>(dev, ws, io, n);
    }
    else k_grad<<<(n + kGradBlock - 1) / kGradBlock, kGradBlock, 0, s>>>(dev, ws, io);
  }
  CUDA_TRY(cudaGetLastError());
#if DR_CHECKS
  if (wave) {   // checked build: every queue entry that was reserved was consumed, every path finished, no check fired
    uint32_t h[kCtlWords];
    CUDA_TRY(cudaMemcpyAsync(h, ws.ctl, sizeof(h), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    if (h[kCtlWaveError] || h[kCtlWaveDone] != n || h[kCtlWaveReserve] > wave_ring_entries(dev, ws.cap))   // with next-event estimation up to (2L - 1) entries per state
      return fail(DR_ERR_CUDA, "k_wave protocol check failed: error bits " + std::to_string(h[kCtlWaveError]) + ", finished " +
                                   std::to_string(h[kCtlWaveDone]) + " of " + std::to_string(n));
  }
#endif
  return DR_OK;
}

// Every evaluation of a chain ensemble gets its own tag (dr_wave.cuh): the state memory is zeroed by dr_chains_init and
// tags start at 1, so queue entries of earlier evaluations never look published.
EvalWs next_ws(dr_chains* c, cudaStream_t s) {
  if (++c->eval_tag == 0) {   // 2^32 evaluations later: clear the queue once and start over
    cudaMemsetAsync(c->ws.ring, 0, sizeof(uint2) * wave_ring_entries(c->scene->dev, c->ws.cap), s);
    c->eval_tag = 1;
  }
  EvalWs ws = c->ws;
  ws.tag = c->eval_tag;
  return ws;
}

EvalIO chain_io(const dr_chains* c, bool use_order) {
  EvalIO io{};
  io.x = c->st.y; io.stride = c->cp.N; io.order = use_order ? c->st.order : nullptr;
  io.g = c->st.gy; io.f = c->st.fy; io.pix = c->st.pixy; io.sig = c->st.sigy; io.nrays = nullptr;
  io.rays_ctr = &c->st.ctr->rays; io.nonfinite_ctr = &c->st.ctr->nonfinite; io.work = nullptr; io.grad_ctr = &c->st.ctr->grad_states;
  return io;
}

// one iteration of every chain: propose, evaluate the proposals, (bootstrap,) decide, compact
dr_status launch_iteration(dr_chains* c, uint32_t n, bool init, cudaStream_t s) {
  const ChainParams& cp = c->cp;
  const uint32_t gb = c->nblocks;
  { ProfScope ps(c, DR_PROF_PROPOSE, s); k_propose<<<gb, kBlock, 0, s>>>(cp, c->st, n, init ? 1 : 0); }
  // evaluation order: alive chains first, then the regeneration queue (a9), once the queue exists
  const dr_status es = launch_eval(c, c->scene, next_ws(c, s), chain_io(c, !init && cp.restore), cp.N, cp.grad != 0, false, c->eval_form, s);
  if (es != DR_OK) return es;
  if (init) {
    k_psum_partial<<<gb, kBlock, 0, s>>>(cp, c->st);
    k_bootstrap<<<1, kBlock, 0, s>>>(cp, c->st, gb);
  }
  { ProfScope ps(c, DR_PROF_DECIDE, s); k_decide<<<gb, kBlock, 0, s>>>(cp, c->st, c->accum, n, c->ws.ctl); }
  if (cp.restore) {
    { ProfScope ps(c, DR_PROF_SCAN, s); k_scan<<<1, 1024, 0, s>>>(c->st, gb); }
    { ProfScope ps(c, DR_PROF_SCATTER, s); k_scatter<<<gb, kBlock, 0, s>>>(cp, c->st); }
  }
  CUDA_TRY(cudaGetLastError());
  return DR_OK;
}

// Device scratch of the test hooks (freed on scope exit).
struct DevBuf {
  void* p = nullptr;
  cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 16); }
  ~DevBuf() { cudaFree(p); }
  template <class T> T* as() const { return (T*)p; }
};

// Workspace + plane buffers for evaluating n states outside a chain ensemble.
struct HookEval {
  DevBuf ws_mem, xpl, gpl, f4;
  EvalWs ws{};
  cudaError_t setup(const dr_scene* sc, uint32_t n, bool grad, cudaStream_t stream) {
    const size_t N = n, L = sc->dev.L;
    size_t o = 0;
    auto take = [&](size_t bytes) { const size_t at = o; o = align256(o + bytes); return at; };
    const bool gn = grad && sc->dev.nee;
    const size_t q = take(96 * N), hits = take(8 * N), ring = take(8 * wave_ring_entries(sc->dev, N)), rec = take(grad ? 16 * N * (gn ? 1 : L) : 0),
                 vrec = take(gn ? 48 * N * L : 0), adj = take(gn ? 48 * N : 0),
                 pinfo = take(grad ? 4 * N : 0), gl = take(grad ? 4 * N * (sc->dev.nee ? 3 * L : 1) : 0), ctl = take(4 * kCtlWords);
    cudaError_t e = ws_mem.alloc(o);
    if (e == cudaSuccess) e = xpl.alloc(16 * N * sc->dev.planes);
    if (e == cudaSuccess) e = gpl.alloc(grad ? 16 * N * sc->dev.planes : 0);
    if (e == cudaSuccess) e = f4.alloc(16 * N);
    if (e != cudaSuccess) return e;
    char* b = ws_mem.as<char>();
    ws.qa = (float4*)(b + q); ws.qb = ws.qa + 3 * N; ws.hits = (uint2*)(b + hits); ws.ring = (uint2*)(b + ring); ws.rec = (float4*)(b + rec);
    ws.vrec = (float4*)(b + vrec); ws.adj = (float4*)(b + adj);
    ws.pinfo = grad ? (uint32_t*)(b + pinfo) : nullptr; ws.gradlist = (uint32_t*)(b + gl); ws.ctl = (uint32_t*)(b + ctl); ws.cap = n;
    ws.tag = 1;
    return cudaMemsetAsync(ws.ring, 0, 8 * wave_ring_entries(sc->dev, N), stream);   // fresh memory: no entry carries tag 1
  }
};

}  // namespace

extern "C" {

const char* dr_last_error(void) { return g_err.c_str(); }

dr_status dr_scene_create(const dr_scene_desc* d, dr_scene** out) {
  if (!d || !out) return fail(DR_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (!d->host_vertices || !d->host_indices || !d->host_tri_material || !d->host_materials)
    return fail(DR_ERR_INVALID_ARG, "null array in scene description");
  if (d->nv < 3 || d->nt < 1 || d->nm < 1) return fail(DR_ERR_INVALID_ARG, "empty scene");
  if (d->nt >= (1u << 27)) return fail(DR_ERR_UNSUPPORTED, "more than 2^27 triangles");
  if (d->width < 1 || d->height < 1) return fail(DR_ERR_INVALID_ARG, "image size must be >= 1");
  if (d->max_path_len < 1 || d->max_path_len > (uint32_t)kMaxPathLen) return fail(DR_ERR_INVALID_ARG, "max_path_len must be in [1,16]");
  if (!(d->vfov_deg > 0.f && d->vfov_deg < 180.f)) return fail(DR_ERR_INVALID_ARG, "vfov_deg must be in (0,180)");
  for (size_t i = 0; i < 3 * (size_t)d->nv; ++i)
    if (!std::isfinite(d->host_vertices[i])) return fail(DR_ERR_NONFINITE, "non-finite vertex");
  for (size_t i = 0; i < 3 * (size_t)d->nt; ++i)
    if (d->host_indices[i] >= d->nv) return fail(DR_ERR_INVALID_ARG, "vertex index out of range");
  for (uint32_t i = 0; i < d->nt; ++i)
    if (d->host_tri_material[i] >= d->nm) return fail(DR_ERR_INVALID_ARG, "material index out of range");
  if (!finite3(d->env_radiance) || !finite3(d->cam_pos) || !finite3(d->cam_look) || !finite3(d->cam_up))
    return fail(DR_ERR_NONFINITE, "non-finite camera or environment");
  std::vector<MatPacked> mats(d->nm);
  for (uint32_t i = 0; i < d->nm; ++i) {
    const dr_material& m = d->host_materials[i];
    if (m.kind < 0 || m.kind > 3) return fail(DR_ERR_INVALID_ARG, "material kind out of range");
    if (!finite3(m.albedo_or_f0) || !finite3(m.emission) || !std::isfinite(m.ior) || !std::isfinite(m.roughness))
      return fail(DR_ERR_NONFINITE, "non-finite material");
    if (m.kind == DR_MAT_DIELECTRIC && !(m.ior > 0.f)) return fail(DR_ERR_INVALID_ARG, "dielectric ior must be > 0");
    if (m.kind == DR_MAT_GGX_CONDUCTOR && !(m.roughness > 0.f && m.roughness <= 1.f))
      return fail(DR_ERR_INVALID_ARG, "GGX roughness must be in (0,1]");
    MatPacked& p = mats[i];
    std::memset(&p, 0, sizeof(p));
    p.kind = (uint32_t)m.kind;
    for (int c = 0; c < 3; ++c) p.a[c] = m.albedo_or_f0[c];
    p.ior = m.ior; p.alpha = m.roughness; p.le0 = m.emission[0]; p.le1 = m.emission[1]; p.le2 = m.emission[2];
  }
  BuiltBvh bvh;
  build_bvh8(d->host_vertices, d->nv, d->host_indices, d->nt, d->host_tri_material, bvh);
  if (bvh.depth > (uint32_t)kMaxBvhDepth) return fail(DR_ERR_UNSUPPORTED, "BVH8 deeper than the traversal stack allows");
  if (bvh.tris.size() >= (size_t(1) << 27))   // k_wave's payload has 27 bits for a state, the vertex record 30 for a triangle reference
    return fail(DR_ERR_UNSUPPORTED, "more than 2^27 triangle references");

  dr_scene* s = new dr_scene();
  DevScene& dev = s->dev;
  const size_t nb = bvh.nodes.size() * sizeof(NodeC), tb = bvh.tris.size() * sizeof(TriPacked), mb = mats.size() * sizeof(MatPacked);
  cudaError_t e = cudaMalloc(&s->d_nodes, nb);
  if (e == cudaSuccess) e = cudaMalloc(&s->d_tris, tb);
  if (e == cudaSuccess) e = cudaMalloc(&s->d_mats, mb);
  if (e == cudaSuccess) e = cudaMemcpy(s->d_nodes, bvh.nodes.data(), nb, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(s->d_tris, bvh.tris.data(), tb, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(s->d_mats, mats.data(), mb, cudaMemcpyHostToDevice);
  int device = 0;
  if (e == cudaSuccess) e = cudaGetDevice(&device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&s->n_sm, cudaDevAttrMultiProcessorCount, device);
  if (e != cudaSuccess) {
    cudaFree(s->d_nodes); cudaFree(s->d_tris); cudaFree(s->d_mats);
    delete s;
    return fail(e == cudaErrorMemoryAllocation ? DR_ERR_OOM : DR_ERR_CUDA, std::string("scene upload: ") + cudaGetErrorString(e));
  }
  dev.nodes = (const uint4*)s->d_nodes; dev.tris = (const float4*)s->d_tris; dev.mats = (const float4*)s->d_mats;
  dev.n_nodes = (uint32_t)bvh.nodes.size();
  dev.stack_cap = bvh.depth + 1;  // node groups: at most one per level
  const size_t stack_bytes = trace_stack_bytes(dev.stack_cap, std::max(kTraceBlock, TraceSmall::kBlock));
  if (stack_bytes > kMaxDynSmem) {   // (depth + 1) node groups per thread no longer fit the block's shared memory
    dr_scene_destroy(s);
    return fail(DR_ERR_UNSUPPORTED, "BVH8 deeper than the traversal stack allows");
  }
  s->trace_smem = trace_stack_bytes(dev.stack_cap, kTraceBlock);
  s->wave_ok = stack_bytes + kWaveExtraSmem <= kMaxDynSmem;
  if (d->nee && !s->wave_ok) {   // next-event estimation has no per-segment loop to fall back on: refuse here, not at the first evaluation
    dr_scene_destroy(s);
    return fail(DR_ERR_UNSUPPORTED, "next-event estimation runs in k_wave only, and this BVH8 is too deep for k_wave's shared memory");
  }
  e = cudaFuncSetAttribute(k_trace<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_trace<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxDynSmem);
  if (e == cudaSuccess) e = wave_allow_smem<TraceBig>();
  if (e == cudaSuccess) e = wave_allow_smem<TraceSmall>();
  if (e != cudaSuccess) {
    dr_scene_destroy(s);
    return fail(DR_ERR_CUDA, std::string("k_trace shared memory: ") + cudaGetErrorString(e));
  }
  dev.n_tris = d->nt; dev.n_mats = d->nm;
  for (int c = 0; c < 3; ++c) { dev.env[c] = d->env_radiance[c]; dev.cam_pos[c] = d->cam_pos[c]; }
  // pinhole basis: w = normalize(look - pos), r = normalize(w x up), v = r x w
  float w[3] = {d->cam_look[0] - d->cam_pos[0], d->cam_look[1] - d->cam_pos[1], d->cam_look[2] - d->cam_pos[2]};
  normalize(w);
  float r[3], v[3];
  cross(w, d->cam_up, r);
  normalize(r);
  cross(r, w, v);
  if (!finite3(w) || !finite3(r)) {
    dr_scene_destroy(s);
    return fail(DR_ERR_INVALID_ARG, "degenerate camera (look == pos or up parallel to view)");
  }
  for (int c = 0; c < 3; ++c) { dev.cam_w[c] = w[c]; dev.cam_r[c] = r[c]; dev.cam_v[c] = v[c]; }
  dev.tan_half = std::tan(d->vfov_deg * (float)(3.14159265358979323846 / 360.0));
  dev.tan_half_aspect = dev.tan_half * ((float)d->width / (float)d->height);
  dev.nee = d->nee ? 1u : 0u;
  dev.W = d->width; dev.H = d->height; dev.L = d->max_path_len; dev.d = (dev.nee ? 4 : 2) * d->max_path_len; dev.planes = (dev.d + 3) / 4;
  // emitter list for next-event estimation (dr_nee.cuh Light; Q21): triangle-index order, areas and running sums in fp32
  {
    std::vector<float> lights;
    float total = 0.f;
    for (uint32_t t = 0; t < d->nt; ++t) {
      const dr_material& m = d->host_materials[d->host_tri_material[t]];
      if (m.kind != DR_MAT_EMITTER) continue;
      const float* a = &d->host_vertices[3 * d->host_indices[3 * t]];
      const float* b = &d->host_vertices[3 * d->host_indices[3 * t + 1]];
      const float* c = &d->host_vertices[3 * d->host_indices[3 * t + 2]];
      float e1[3], e2[3], cr[3];
      for (int x = 0; x < 3; ++x) { e1[x] = b[x] - a[x]; e2[x] = c[x] - a[x]; }
      cross(e1, e2, cr);
      const float area = 0.5f * std::sqrt(cr[0] * cr[0] + cr[1] * cr[1] + cr[2] * cr[2]);
      if (!(area > 0.f) || !std::isfinite(area)) continue;   // a degenerate emitter has no normal and no area to sample: it is never picked (nor can a ray hit it)
      const float before = total;
      total = total + area;
      normalize(cr);
      uint32_t idbits = t;
      float idf;
      std::memcpy(&idf, &idbits, 4);
      const float rec[20] = {a[0], a[1], a[2], total, e1[0], e1[1], e1[2], area, e2[0], e2[1], e2[2], idf,
                             cr[0], cr[1], cr[2], before, m.emission[0], m.emission[1], m.emission[2], 0.f};
      lights.insert(lights.end(), rec, rec + 20);
    }
    if (!(total > 0.f) || !std::isfinite(total)) lights.clear();   // no emitter area to sample: vertices make no emitter connection (dr_nee.cuh checks n_lights)
    dev.n_lights = (uint32_t)(lights.size() / 20);
    dev.light_total = dev.n_lights ? total : 0.f;
    dev.lights = nullptr;
    if (dev.n_lights) {
      cudaError_t le = cudaMalloc(&s->d_lights, lights.size() * sizeof(float));
      if (le == cudaSuccess) le = cudaMemcpy(s->d_lights, lights.data(), lights.size() * sizeof(float), cudaMemcpyHostToDevice);
      if (le != cudaSuccess) { dr_scene_destroy(s); return fail(DR_ERR_CUDA, std::string("emitter list: ") + cudaGetErrorString(le)); }
      dev.lights = (const float4*)s->d_lights;
    }
  }
  dev.eps_ray = 1e-5f * bvh.diag;  // Q8
  dev.analytic = 0; dev.n_mix = 0;
  s->info.n_tris = d->nt; s->info.n_nodes = dev.n_nodes; s->info.depth = bvh.depth; s->info.smem_nodes = 0;
  s->info.sah_cost = bvh.sah_cost; s->info.eps_ray = dev.eps_ray; s->info.device_bytes = nb + tb + mb;
  *out = s;
  return DR_OK;
}

dr_status dr_scene_create_analytic2d(const dr_analytic2d_desc* d, dr_scene** out) {
  if (!d || !out) return fail(DR_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (d->n_components < 1 || d->n_components > (uint32_t)kMaxMix) return fail(DR_ERR_INVALID_ARG, "n_components must be in [1,16]");
  if (!d->host_weights || !d->host_means || !d->host_stddevs) return fail(DR_ERR_INVALID_ARG, "null array");
  if (d->width < 1 || d->height < 1) return fail(DR_ERR_INVALID_ARG, "image size must be >= 1");
  dr_scene* s = new dr_scene();
  DevScene& dev = s->dev;
  for (uint32_t k = 0; k < d->n_components; ++k) {
    const float w = d->host_weights[k], sd = d->host_stddevs[k], mx = d->host_means[2 * k], my = d->host_means[2 * k + 1];
    if (!(std::isfinite(w) && std::isfinite(sd) && std::isfinite(mx) && std::isfinite(my))) { delete s; return fail(DR_ERR_NONFINITE, "non-finite mixture parameter"); }
    if (!(w > 0.f) || !(sd > 0.f)) { delete s; return fail(DR_ERR_INVALID_ARG, "weights and stddevs must be > 0"); }
    dev.mix_w[k] = w; dev.mix_s[k] = sd; dev.mix_mx[k] = mx; dev.mix_my[k] = my;
  }
  dev.analytic = 1; dev.n_mix = (int)d->n_components;
  dev.W = d->width; dev.H = d->height; dev.L = 1; dev.d = 2; dev.planes = 1;
  dev.n_nodes = 0; dev.nee = 0; dev.n_lights = 0; dev.lights = nullptr; dev.light_total = 0.f;
  s->info = dr_scene_info{};
  *out = s;
  return DR_OK;
}

dr_status dr_scene_destroy(dr_scene* s) {
  if (!s) return DR_OK;
  cudaFree(s->d_nodes); cudaFree(s->d_tris); cudaFree(s->d_mats); cudaFree(s->d_lights);
  delete s;
  return DR_OK;
}

dr_status dr_scene_get_info(const dr_scene* s, dr_scene_info* o) {
  if (!s || !o) return fail(DR_ERR_INVALID_ARG, "null argument");
  *o = s->info;
  return DR_OK;
}

dr_status dr_config_default(int32_t method, double stddev, dr_config* out) {
  if (!out) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (method < 0 || method > DR_PATH_TRACING) return fail(DR_ERR_INVALID_ARG, "method out of range");
  if (!std::isfinite(stddev)) return fail(DR_ERR_INVALID_ARG, "stddev must be finite");
  std::memset(out, 0, sizeof(*out));
  const bool random_walk = method == DR_METROPOLIS || method == DR_METROPOLIS_RESTORE;
  const double s = stddev > 0.0 ? stddev : (random_walk ? 1e-2 : 5e-3);
  out->method = method;
  out->stddev = (float)s;
  out->c_tilde = (float)(0.5 * s * s);                                                                  // DESIGN.md Q10, in double like the caller's own s^2 / 2 would be
  out->dt = 1e-5f;                                                                                      // L755
  out->m = 64.f;                                                                                        // L754
  out->large_step_prob = (method == DR_METROPOLIS || method == DR_MALA) ? 0.3f : 0.f;                   // L747
  return DR_OK;
}

size_t dr_chains_state_bytes(const dr_scene* s, const dr_config* c) {
  if (!s || check_config(c) != DR_OK) return 0;
  const bool grad = c->method == DR_MALA || c->method == DR_MALA_RESTORE || c->method == DR_DIFFUSION_RESTORE;
  return make_layout(c->n_chains, s->dev.planes, s->dev.L, grad, s->dev.nee != 0).total;
}

dr_status dr_chains_create(const dr_scene* s, const dr_config* c, void* dev_state, size_t bytes, float* dev_accum, dr_chains** out) {
  if (!s || !out || !dev_state || !dev_accum) return fail(DR_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  const dr_status cs = check_config(c);
  if (cs != DR_OK) return cs;
  if (((uintptr_t)dev_state & 255u) || ((uintptr_t)dev_accum & 15u)) return fail(DR_ERR_INVALID_ARG, "dev_state must be 256-byte and dev_accum 16-byte aligned");
  const bool grad = c->method == DR_MALA || c->method == DR_MALA_RESTORE || c->method == DR_DIFFUSION_RESTORE;
  const Layout L = make_layout(c->n_chains, s->dev.planes, s->dev.L, grad, s->dev.nee != 0);
  if (bytes < L.total) return fail(DR_ERR_INVALID_ARG, "state buffer smaller than dr_chains_state_bytes");
  dr_chains* h = new dr_chains();
  h->scene = s; h->cfg = *c;
  ChainParams& cp = h->cp;
  cp.method = c->method; cp.restore = c->method >= DR_METROPOLIS_RESTORE && c->method <= DR_DIFFUSION_RESTORE; cp.grad = grad;
  cp.rao_blackwell = cp.restore && c->rao_blackwell;
  cp.a_mode = (int)c->a_mode; cp.rho_grid = c->rho_grid; cp.rho = nullptr;
  if (c->rho_grid) {   // running sums in fp32, in tile order (what the regeneration inverts)
    std::vector<float> t2(2 * (size_t)c->rho_grid * c->rho_grid);
    float acc = 0.f;
    for (uint32_t t = 0; t < c->rho_grid * c->rho_grid; ++t) { acc = acc + c->host_rho[t]; t2[2 * t] = c->host_rho[t]; t2[2 * t + 1] = acc; }
    cudaError_t re = cudaMalloc(&h->d_rho, t2.size() * sizeof(float));
    if (re == cudaSuccess) re = cudaMemcpy(h->d_rho, t2.data(), t2.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (re != cudaSuccess) { delete h; return fail(DR_ERR_CUDA, std::string("regeneration density: ") + cudaGetErrorString(re)); }
    cp.rho = (const float2*)h->d_rho;
    h->cfg.host_rho = nullptr;   // the caller's array is not kept
  }
  cp.N = c->n_chains; cp.d = s->dev.d; cp.planes = s->dev.planes;
  cp.stddev = c->stddev; cp.half_s2 = 0.5f * c->stddev * c->stddev; cp.c_tilde = c->c_tilde; cp.dt = c->dt; cp.m = c->m;
  cp.large_step_prob = cp.restore ? 0.f : c->large_step_prob;
  cp.p_lambda_override = c->p_lambda_override; cp.seed = c->seed; cp.epoch = 0; cp.chain_offset = c->chain_offset;
  char* b = (char*)dev_state;
  ChainState& st = h->st;
  st.x = (float4*)(b + L.x); st.g = (float4*)(b + L.g); st.fp = (float4*)(b + L.fp); st.pix = (uint32_t*)(b + L.pix);
  st.sig = (uint32_t*)(b + L.sig); st.killed = (uint8_t*)(b + L.killed); st.y = (float4*)(b + L.y); st.gy = (float4*)(b + L.gy);
  st.fy = (float4*)(b + L.fy); st.pixy = (uint32_t*)(b + L.pixy); st.sigy = (uint32_t*)(b + L.sigy); st.kind = (uint8_t*)(b + L.kind);
  st.accepted = (uint8_t*)(b + L.accepted); st.weight = (float*)(b + L.weight); st.order = (uint32_t*)(b + L.order);
  st.blockcnt = (uint32_t*)(b + L.blockcnt); st.blockoff = (uint32_t*)(b + L.blockoff); st.partial = (double*)(b + L.partial);
  st.ctr = (Counters*)(b + L.ctr);
  h->accum = (float4*)dev_accum;
  h->npix = s->dev.W * s->dev.H;
  h->nblocks = (cp.N + kBlock - 1) / kBlock;
  h->state_bytes = L.total; h->state_base = dev_state;
  EvalWs& ws = h->ws;
  ws.qa = (float4*)(b + L.q); ws.qb = ws.qa + 3 * (size_t)cp.N; ws.hits = (uint2*)(b + L.hits); ws.ring = (uint2*)(b + L.ring);
  ws.rec = (float4*)(b + L.rec); ws.vrec = (float4*)(b + L.vrec); ws.adj = (float4*)(b + L.adj);
  ws.pinfo = cp.grad ? (uint32_t*)(b + L.pinfo) : nullptr; ws.gradlist = (uint32_t*)(b + L.gradlist); ws.ctl = (uint32_t*)(b + L.ctl); ws.cap = cp.N;
  if (cudaHostAlloc((void**)&h->h_last_rays, sizeof(uint32_t), cudaHostAllocDefault) == cudaSuccess) *h->h_last_rays = 0u;
  else { h->h_last_rays = nullptr; (void)cudaGetLastError(); }   // only a hint: without it the shape goes by the number of states
  *out = h;
  return DR_OK;
}

dr_status dr_chains_destroy(dr_chains* c) { delete c; return DR_OK; }

dr_status dr_chains_set_eval_form(dr_chains* c, int32_t form) {
  if (!c) return fail(DR_ERR_INVALID_ARG, "null chains");
  if (form < 0 || form > 4) return fail(DR_ERR_INVALID_ARG, "form must be 0 .. 4");
  c->eval_form = form;
  return DR_OK;
}

dr_status dr_chains_init(dr_chains* c, uint32_t frame_index, void* stream) {
  if (!c) return fail(DR_ERR_INVALID_ARG, "null chains");
  if (frame_index >= (1u << 24)) return fail(DR_ERR_INVALID_ARG, "frame_index must be < 2^24");
  cudaStream_t s = (cudaStream_t)stream;
  c->cp.epoch = frame_index;
  c->iteration = 0;
  CUDA_TRY(cudaMemsetAsync(c->state_base, 0, c->state_bytes, s));
  CUDA_TRY(cudaMemsetAsync(c->accum, 0, sizeof(float4) * (size_t)c->npix, s));
  const dr_status r = launch_iteration(c, 0, true, s);
  if (r == DR_OK) c->initialised = true;
  return r;
}

dr_status dr_step(dr_chains* c, int32_t method, uint32_t iterations, void* stream) {
  if (!c) return fail(DR_ERR_INVALID_ARG, "null chains");
  if (method != c->cfg.method) return fail(DR_ERR_INVALID_ARG, "method differs from the one the chains were created with");
  if (!c->initialised) return fail(DR_ERR_INVALID_ARG, "dr_chains_init has not been called");
  for (uint32_t k = 0; k < iterations; ++k) {
    const dr_status r = launch_iteration(c, ++c->iteration, false, (cudaStream_t)stream);
    if (r != DR_OK) return r;
  }
  return DR_OK;
}

dr_status dr_resolve_image(dr_chains* c, float* dev_rgb, void* stream) {
  if (!c || !dev_rgb) return fail(DR_ERR_INVALID_ARG, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  { ProfScope ps(c, DR_PROF_RESOLVE, s); k_resolve<<<(c->npix + kBlock - 1) / kBlock, kBlock, 0, s>>>(c->cp, c->st.ctr, c->accum, dev_rgb, c->npix, 0ull, 0ull, nullptr); }
  CUDA_TRY(cudaGetLastError());
  return DR_OK;   // asynchronous: a resolve before the first completed tour writes zeros and is counted (dr_stats.no_tour_resolves)
}

dr_status dr_resolve_image_sharded(dr_chains* c, const float* dev_accum_sum, uint64_t tours_total, uint64_t mutations_total,
                                   float* dev_rgb, void* stream) {
  if (!c || !dev_rgb || !dev_accum_sum) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (!mutations_total) return fail(DR_ERR_INVALID_ARG, "mutations_total must be > 0");
  {
    ProfScope ps(c, DR_PROF_RESOLVE, (cudaStream_t)stream);
    k_resolve<<<(c->npix + kBlock - 1) / kBlock, kBlock, 0, (cudaStream_t)stream>>>(
        c->cp, c->st.ctr, (const float4*)dev_accum_sum, dev_rgb, c->npix, (unsigned long long)tours_total,
        (unsigned long long)mutations_total, nullptr);
  }
  CUDA_TRY(cudaGetLastError());
  return DR_OK;
}

size_t dr_frame_floats(const dr_chains* c) { return c ? 4 * (size_t)c->npix + kTailFloats : 0; }

dr_status dr_pack_frame(dr_chains* c, float* dev_buf, void* stream) {
  if (!c || !dev_buf) return fail(DR_ERR_INVALID_ARG, "null argument");
  if ((uintptr_t)dev_buf & 15u) return fail(DR_ERR_INVALID_ARG, "dev_buf must be 16-byte aligned");
  k_pack_frame<<<(c->npix + kBlock - 1) / kBlock, kBlock, 0, (cudaStream_t)stream>>>(c->st.ctr, c->accum, dev_buf, c->npix);
  CUDA_TRY(cudaGetLastError());
  return DR_OK;
}

dr_status dr_resolve_image_packed(dr_chains* c, const float* dev_buf_sum, float* dev_rgb, void* stream) {
  if (!c || !dev_rgb || !dev_buf_sum) return fail(DR_ERR_INVALID_ARG, "null argument");
  if ((uintptr_t)dev_buf_sum & 15u) return fail(DR_ERR_INVALID_ARG, "dev_buf_sum must be 16-byte aligned");
  {
    ProfScope ps(c, DR_PROF_RESOLVE, (cudaStream_t)stream);
    k_resolve<<<(c->npix + kBlock - 1) / kBlock, kBlock, 0, (cudaStream_t)stream>>>(
        c->cp, c->st.ctr, (const float4*)dev_buf_sum, dev_rgb, c->npix, 0ull, 0ull, dev_buf_sum + 4 * (size_t)c->npix);
  }
  CUDA_TRY(cudaGetLastError());
  return DR_OK;
}

dr_status dr_profile_enable(dr_chains* c, int32_t on, void* stream) {
  if (!c) return fail(DR_ERR_INVALID_ARG, "null chains");
  CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
  prof_drain(c);
  for (int k = 0; k < DR_PROF_COUNT; ++k) { c->prof_ms[k] = 0; c->prof_launches[k] = 0; }
  c->profiling = on != 0;
  return DR_OK;
}

dr_status dr_profile_read(dr_chains* c, double* host_ms, uint64_t* host_launches, void* stream) {
  if (!c || !host_ms || !host_launches) return fail(DR_ERR_INVALID_ARG, "null argument");
  CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
  prof_drain(c);
  for (int k = 0; k < DR_PROF_COUNT; ++k) { host_ms[k] = c->prof_ms[k]; host_launches[k] = c->prof_launches[k]; }
  return DR_OK;
}

dr_status dr_chains_work_stats(dr_chains* c, uint64_t* host_out3, void* stream) {
  if (!c || !host_out3) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (!c->initialised) return fail(DR_ERR_INVALID_ARG, "dr_chains_init has not been called");
  cudaStream_t s = (cudaStream_t)stream;
  DevBuf d;
  CUDA_TRY(d.alloc(24));
  CUDA_TRY(cudaMemsetAsync(d.p, 0, 24, s));
  // re-evaluates the last proposals (same values are written again) with the counting variant of k_trace
  EvalIO io = chain_io(c, false);
  io.rays_ctr = d.as<unsigned long long>(); io.nonfinite_ctr = nullptr; io.work = d.as<unsigned long long>() + 1; io.grad_ctr = nullptr;
  if (c->cp.grad) CUDA_TRY(cudaMemsetAsync(c->st.gy, 0, sizeof(float4) * (size_t)c->cp.planes * c->cp.N, s));
  const dr_status r = launch_eval(nullptr, c->scene, next_ws(c, s), io, c->cp.N, c->cp.grad != 0, true, 0, s);
  if (r != DR_OK) return r;
  CUDA_TRY(cudaMemcpyAsync(host_out3, d.p, 24, cudaMemcpyDeviceToHost, s));
  uint32_t wave_err = 0;
  if (!c->scene->dev.analytic) CUDA_TRY(cudaMemcpyAsync(&wave_err, c->ws.ctl + kCtlWaveError, 4, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));
  if (wave_err & kErrTimeout) return fail(DR_ERR_CUDA, "k_wave's watchdog ended the counting evaluation: the counts are incomplete");
  return DR_OK;
}

dr_status dr_chains_stats(dr_chains* c, dr_stats* o, void* stream) {
  if (!c || !o) return fail(DR_ERR_INVALID_ARG, "null argument");
  Counters h;
  CUDA_TRY(cudaMemcpyAsync(&h, c->st.ctr, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
  o->tours = h.tours; o->mutations = h.mutations; o->rays = h.rays; o->mh_accepts = h.mh_accepts; o->nonfinite = h.nonfinite;
  o->kills_last_step = h.kills_last; o->regen_queue_len = h.queue_len; o->iteration = c->iteration;
  o->p_lambda = h.p_lambda; o->kappa0 = h.kappa0; o->lambda = h.lambda; o->no_tour_resolves = h.no_tour_resolves;
  o->grad_states = h.grad_states; o->lit_init = h.lit_init; o->wave_timeouts = h.wave_timeouts;
  if (h.wave_timeouts) return fail(DR_ERR_CUDA, "k_wave's watchdog ended an evaluation: results since dr_chains_init are invalid");
  if (h.no_tour_resolves) { g_err = "a resolve ran before any tour had completed: zero image"; return DR_WARN_NO_TOURS; }
  return DR_OK;
}

// ---- test hooks ---------------------------------------------------------------------------------------------
// Staging layout of the two hooks: x rows | score rows | p | f/p_hat   (N * (8 d + 16) bytes, kept for the life of the chains)
namespace {
struct HookStage { float *x, *g, *p, *fop; };
dr_status hook_stage(dr_chains* c, HookStage& st) {
  const size_t N = c->cp.N, d = c->cp.d;
  if (!c->hook_scratch) CUDA_TRY(cudaMalloc(&c->hook_scratch, sizeof(float) * N * (2 * d + 4)));
  st.x = (float*)c->hook_scratch; st.g = st.x + N * d; st.p = st.g + N * d; st.fop = st.p + N;
  return DR_OK;
}
}  // namespace

dr_status dr_chains_download(dr_chains* c, float* hx, float* hp, float* hfop, uint32_t* hpix, uint8_t* hkilled, float* hscore,
                             uint32_t* hsig, void* stream) {
  if (!c) return fail(DR_ERR_INVALID_ARG, "null chains");
  cudaStream_t s = (cudaStream_t)stream;
  const uint32_t N = c->cp.N, d = c->cp.d, g = (N + 255) / 256;
  HookStage st;
  const dr_status rs = hook_stage(c, st);
  if (rs != DR_OK) return rs;
  // every conversion kernel and copy is queued on the stream; one synchronisation at the end (pinned host arrays copy by DMA)
  if (hx) { k_planes_to_rows<<<g, 256, 0, s>>>(c->st.x, st.x, N, d, c->cp.planes); CUDA_TRY(cudaMemcpyAsync(hx, st.x, sizeof(float) * (size_t)N * d, cudaMemcpyDeviceToHost, s)); }
  if (hscore && c->cp.grad) { k_planes_to_rows<<<g, 256, 0, s>>>(c->st.g, st.g, N, d, c->cp.planes); CUDA_TRY(cudaMemcpyAsync(hscore, st.g, sizeof(float) * (size_t)N * d, cudaMemcpyDeviceToHost, s)); }
  if (hp || hfop) k_fp_split<<<g, 256, 0, s>>>(c->st.fp, hp ? st.p : nullptr, hfop ? st.fop : nullptr, N);
  if (hp) CUDA_TRY(cudaMemcpyAsync(hp, st.p, 4 * (size_t)N, cudaMemcpyDeviceToHost, s));
  if (hfop) CUDA_TRY(cudaMemcpyAsync(hfop, st.fop, 12 * (size_t)N, cudaMemcpyDeviceToHost, s));
  if (hpix) CUDA_TRY(cudaMemcpyAsync(hpix, c->st.pix, 4 * (size_t)N, cudaMemcpyDeviceToHost, s));
  if (hsig) CUDA_TRY(cudaMemcpyAsync(hsig, c->st.sig, 4 * (size_t)N, cudaMemcpyDeviceToHost, s));
  if (hkilled) CUDA_TRY(cudaMemcpyAsync(hkilled, c->st.killed, N, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaStreamSynchronize(s));
  if (hscore && !c->cp.grad) std::memset(hscore, 0, sizeof(float) * (size_t)N * d);
  return DR_OK;
}

dr_status dr_chains_upload(dr_chains* c, const float* hx, const float* hp, const float* hfop, const uint32_t* hpix,
                           const uint8_t* hkilled, const float* hscore, const uint32_t* hsig, uint32_t iteration, void* stream) {
  if (!c || !hx || !hp || !hfop || !hpix || !hkilled) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (c->cp.grad && !hscore) return fail(DR_ERR_INVALID_ARG, "score required for gradient methods");
  if (!c->initialised) return fail(DR_ERR_INVALID_ARG, "dr_chains_init has not been called");
  cudaStream_t s = (cudaStream_t)stream;
  const uint32_t N = c->cp.N, d = c->cp.d, g = (N + 255) / 256;
  HookStage st;
  const dr_status rs = hook_stage(c, st);
  if (rs != DR_OK) return rs;
  CUDA_TRY(cudaMemcpyAsync(st.x, hx, sizeof(float) * (size_t)N * d, cudaMemcpyHostToDevice, s));
  k_rows_to_planes<<<g, 256, 0, s>>>(st.x, c->st.x, N, d, c->cp.planes);
  if (c->cp.grad) {
    CUDA_TRY(cudaMemcpyAsync(st.g, hscore, sizeof(float) * (size_t)N * d, cudaMemcpyHostToDevice, s));
    k_rows_to_planes<<<g, 256, 0, s>>>(st.g, c->st.g, N, d, c->cp.planes);
  }
  CUDA_TRY(cudaMemcpyAsync(st.p, hp, 4 * (size_t)N, cudaMemcpyHostToDevice, s));
  CUDA_TRY(cudaMemcpyAsync(st.fop, hfop, 12 * (size_t)N, cudaMemcpyHostToDevice, s));
  k_fp_join<<<g, 256, 0, s>>>(st.p, st.fop, c->st.fp, N);
  CUDA_TRY(cudaMemcpyAsync(c->st.pix, hpix, 4 * (size_t)N, cudaMemcpyHostToDevice, s));
  CUDA_TRY(cudaMemcpyAsync(c->st.killed, hkilled, N, cudaMemcpyHostToDevice, s));
  if (hsig) CUDA_TRY(cudaMemcpyAsync(c->st.sig, hsig, 4 * (size_t)N, cudaMemcpyHostToDevice, s));
  if (c->cp.restore) {
    k_count_killed<<<c->nblocks, kBlock, 0, s>>>(c->cp, c->st);
    k_scan<<<1, 1024, 0, s>>>(c->st, c->nblocks);
    k_scatter<<<c->nblocks, kBlock, 0, s>>>(c->cp, c->st);
  }
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaStreamSynchronize(s));   // the host arrays may be reused on return
  c->iteration = iteration;
  return DR_OK;
}

dr_status dr_chains_last_step(dr_chains* c, uint8_t* hacc, float* hw, void* stream) {
  if (!c) return fail(DR_ERR_INVALID_ARG, "null chains");
  cudaStream_t s = (cudaStream_t)stream;
  if (hacc) CUDA_TRY(cudaMemcpyAsync(hacc, c->st.accepted, c->cp.N, cudaMemcpyDeviceToHost, s));
  if (hw) CUDA_TRY(cudaMemcpyAsync(hw, c->st.weight, 4 * (size_t)c->cp.N, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));
  return DR_OK;
}

dr_status dr_regen_queue_download(dr_chains* c, uint32_t* hids, uint32_t* hlen, void* stream) {
  if (!c || !hlen) return fail(DR_ERR_INVALID_ARG, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  *hlen = 0;
  if (!c->cp.restore) return DR_OK;
  uint32_t q = 0;
  CUDA_TRY(cudaMemcpyAsync(&q, &c->st.ctr->queue_len, 4, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));
  *hlen = q;
  if (hids && q) {
    CUDA_TRY(cudaMemcpyAsync(hids, c->st.order + (c->cp.N - q), 4 * (size_t)q, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
  }
  return DR_OK;
}

dr_status dr_trace_rays(const dr_scene* sc, const float* o, const float* d, uint32_t n, float* t, uint32_t* prim, void* stream) {
  if (!sc) return fail(DR_ERR_INVALID_ARG, "null scene");
  if (sc->dev.analytic) return fail(DR_ERR_UNSUPPORTED, "analytic scene has no geometry");
  if (!n) return DR_OK;  // empty input: nothing to do, pointers may be null
  if (!o || !d || !t || !prim) return fail(DR_ERR_INVALID_ARG, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  DevBuf q, hits, ctl;
  CUDA_TRY(q.alloc(32 * (size_t)n));
  CUDA_TRY(hits.alloc(8 * (size_t)n));
  CUDA_TRY(ctl.alloc(8));
  CUDA_TRY(cudaMemsetAsync(ctl.p, 0, 8, s));
  const uint32_t g = (n + 255) / 256;
  k_pack_rays<<<g, 256, 0, s>>>(o, d, n, q.as<float4>(), n, ctl.as<uint32_t>());
  k_trace<false><<<sc->n_sm, kTraceBlock, sc->trace_smem, s>>>(sc->dev, q.as<float4>(), n, ctl.as<uint32_t>(), ctl.as<uint32_t>() + 1,
                                                               hits.as<uint2>(), nullptr);
  k_unpack_hits<<<g, 256, 0, s>>>(sc->dev, hits.as<uint2>(), n, t, prim);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaStreamSynchronize(s));  // the scratch buffers are freed on return
  return DR_OK;
}

namespace {
// Evaluates n row-major states through the wavefront path.  Any output may be null.  work3: {rays, nodes, tris} counters.
dr_status eval_rows(const dr_scene* sc, const float* x, uint32_t n, float* f, float* p, uint32_t* pix, float* score, uint32_t* nrays,
                    uint32_t* sig, unsigned long long* work3, int form, cudaStream_t s) {
  const bool grad = score != nullptr;
  const uint32_t d = sc->dev.d, planes = sc->dev.planes, g = (n + 255) / 256;
  HookEval he;
  DevBuf tpix, tsig;
  CUDA_TRY(he.setup(sc, n, grad, s));
  CUDA_TRY(tpix.alloc(4 * (size_t)n));
  CUDA_TRY(tsig.alloc(4 * (size_t)n));
  k_rows_to_planes<<<g, 256, 0, s>>>(x, he.xpl.as<float4>(), n, d, planes);
  if (grad) CUDA_TRY(cudaMemsetAsync(he.gpl.p, 0, 16 * (size_t)n * planes, s));
  EvalIO io{};
  io.x = he.xpl.as<float4>(); io.stride = n; io.order = nullptr; io.g = he.gpl.as<float4>(); io.f = he.f4.as<float4>();
  io.pix = pix ? pix : tpix.as<uint32_t>(); io.sig = sig ? sig : tsig.as<uint32_t>(); io.nrays = nrays;
  io.rays_ctr = work3; io.nonfinite_ctr = nullptr; io.work = work3 ? work3 + 1 : nullptr;
  const dr_status r = launch_eval(nullptr, sc, he.ws, io, n, grad, work3 != nullptr, form, s);
  if (r != DR_OK) return r;
  if (f || p) k_fp_split<<<g, 256, 0, s>>>(he.f4.as<float4>(), p, f, n);
  if (grad) k_planes_to_rows<<<g, 256, 0, s>>>(he.gpl.as<float4>(), score, n, d, planes);
  CUDA_TRY(cudaGetLastError());
  uint32_t wave_err = 0;   // k_wave's watchdog (dr_wave.cuh): an evaluation it ended has written partial results
  if (!sc->dev.analytic) CUDA_TRY(cudaMemcpyAsync(&wave_err, he.ws.ctl + kCtlWaveError, 4, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));  // the scratch buffers are freed on return
  if (wave_err & kErrTimeout) return fail(DR_ERR_CUDA, "k_wave's watchdog ended the evaluation: the outputs are incomplete");
  return DR_OK;
}
}  // namespace

dr_status dr_eval_states(const dr_scene* sc, const float* x, uint32_t n, float* f, float* p, uint32_t* pix, float* score,
                         uint32_t* nrays, uint32_t* sig, void* stream) {
  return dr_eval_states_form(sc, x, n, f, p, pix, score, nrays, sig, 0, stream);
}

dr_status dr_eval_states_form(const dr_scene* sc, const float* x, uint32_t n, float* f, float* p, uint32_t* pix, float* score,
                              uint32_t* nrays, uint32_t* sig, int32_t form, void* stream) {
  if (!sc) return fail(DR_ERR_INVALID_ARG, "null scene");
  if (form < 0 || form > 4) return fail(DR_ERR_INVALID_ARG, "form must be 0 .. 4");
  if (!n) return DR_OK;  // empty input
  if (!x || !f || !p || !pix || !nrays || !sig) return fail(DR_ERR_INVALID_ARG, "null argument");
  return eval_rows(sc, x, n, f, p, pix, score, nrays, sig, nullptr, form, (cudaStream_t)stream);
}

dr_status dr_eval_work_stats(const dr_scene* sc, const float* x, uint32_t n, uint64_t* dev_out3, void* stream) {
  if (!sc) return fail(DR_ERR_INVALID_ARG, "null scene");
  if (!n) return DR_OK;
  if (!x || !dev_out3) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (sc->dev.analytic) return DR_OK;
  return eval_rows(sc, x, n, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, (unsigned long long*)dev_out3, 0, (cudaStream_t)stream);
}

dr_status dr_bias_field(const dr_scene* sc, double stddev, double c_tilde, double dt, uint32_t G, uint32_t M, double* dev_out, void* stream) {
  if (!sc || !dev_out) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (!sc->dev.analytic) return fail(DR_ERR_UNSUPPORTED, "the bias field is defined on the 2-D analytic target");
  if (!(stddev > 0.0) || !(dt > 0.0) || !std::isfinite(c_tilde) || G < 1 || M < 1 || M > 4096) return fail(DR_ERR_INVALID_ARG, "stddev, dt > 0; 1 <= M <= 4096");
  cudaStream_t s = (cudaStream_t)stream;
  DevBuf tab;
  CUDA_TRY(tab.alloc(3 * sizeof(double) * (size_t)M * M));
  k_bias_table<<<(M * M + 255) / 256, 256, 0, s>>>(sc->dev, stddev, c_tilde, M, tab.as<double>());
  k_bias_field<<<G * G, 256, 0, s>>>(sc->dev, stddev, dt, G, M, tab.as<double>(), dev_out);
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaStreamSynchronize(s));   // the table is freed on return
  return DR_OK;
}

dr_status dr_philox_blocks(uint64_t seed, const uint32_t* ctr, uint32_t n, uint32_t* out, void* stream) {
  if (!ctr || !out) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (!n) return DR_OK;
  k_philox_blocks<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(seed, ctr, n, out);
  CUDA_TRY(cudaGetLastError());
  return DR_OK;
}

dr_status dr_rng_transforms(const uint32_t* words, uint32_t n, float* out, void* stream) {
  if (!words || !out) return fail(DR_ERR_INVALID_ARG, "null argument");
  if (!n) return DR_OK;
  k_rng_transforms<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(words, n, out);
  CUDA_TRY(cudaGetLastError());
  return DR_OK;
}

}  // extern "C"

// ---- dr_trace_rays_noalloc (include/dr.h): closest hits without any allocation at call time ---------------------------
// For callers that may not call cudaMalloc / cudaFree when they trace: a frame loop or a server with a fixed memory budget
// (an allocation can fail late, cudaFree stalls the whole device), a host whose own pool already owns the GPU's memory, a
// plugin that must leave its host process's footprint alone.  The kernels are dr_trace_rays' own (k_pack_rays, k_trace,
// k_unpack_hits); only where their scratch lives differs: in this array, which is part of the library image.  Every GPU
// that loads the library carries it (2.5 MiB) until the process ends.
constexpr size_t kNoallocCtlBytes = 256;                                                     // cnt, head (two words) + padding
constexpr size_t kNoallocQueueBytes = 2 * sizeof(float4) * (size_t)DR_TRACE_NOALLOC_MAX_RAYS; // planes o | d
constexpr size_t kNoallocHitsBytes = sizeof(uint2) * (size_t)DR_TRACE_NOALLOC_MAX_RAYS;
constexpr size_t kNoallocBytes = kNoallocCtlBytes + kNoallocQueueBytes + kNoallocHitsBytes;

static __device__ __align__(256) unsigned char g_trace_noalloc_scratch[kNoallocBytes];

namespace {

// In host code the name g_trace_noalloc_scratch is only a handle for the runtime, not a device pointer: a kernel given
// &g_trace_noalloc_scratch[0] from here would fault (or quietly use host memory where the GPU can reach it).  The device
// address comes from cudaGetSymbolAddress, asked once per device with that device current, and is kept here.
constexpr int kNoallocMaxDevices = 64;
unsigned char* g_noalloc_dev_ptr[kNoallocMaxDevices] = {};
std::mutex g_noalloc_mutex;

dr_status noalloc_scratch(unsigned char** out) {
  int device = -1;
  CUDA_TRY(cudaGetDevice(&device));
  if (device < 0 || device >= kNoallocMaxDevices) return fail(DR_ERR_UNSUPPORTED, "dr_trace_rays_noalloc: device ordinal above 63");
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_dev_ptr[device]) {
    void* p = nullptr;
    CUDA_TRY(cudaGetSymbolAddress(&p, g_trace_noalloc_scratch));   // first call on this device: do it before any stream capture
    if (!p) return fail(DR_ERR_CUDA, "dr_trace_rays_noalloc: cudaGetSymbolAddress returned a null address");
    g_noalloc_dev_ptr[device] = static_cast<unsigned char*>(p);
  }
  *out = g_noalloc_dev_ptr[device];
  return DR_OK;
}

}  // namespace

extern "C" dr_status dr_trace_rays_noalloc(const dr_scene* sc, const float* o, const float* d, uint32_t n, float* t, uint32_t* prim,
                                           void* stream) {
  if (!sc) return fail(DR_ERR_INVALID_ARG, "null scene");
  if (sc->dev.analytic) return fail(DR_ERR_UNSUPPORTED, "analytic scene has no geometry");
  if (n > DR_TRACE_NOALLOC_MAX_RAYS)
    return fail(DR_ERR_INVALID_ARG, "dr_trace_rays_noalloc: n = " + std::to_string(n) + " rays exceed the fixed scratch of DR_TRACE_NOALLOC_MAX_RAYS = " +
                                        std::to_string(DR_TRACE_NOALLOC_MAX_RAYS) + " rays; split the batch or use dr_trace_rays");
  if (!n) return DR_OK;  // empty input: nothing to do, pointers may be null
  if (!o || !d || !t || !prim) return fail(DR_ERR_INVALID_ARG, "null argument");
  unsigned char* base = nullptr;
  const dr_status st = noalloc_scratch(&base);
  if (st != DR_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  uint32_t* ctl = reinterpret_cast<uint32_t*>(base);                                   // [0] = ray count, [1] = k_trace's fetch counter
  float4* q = reinterpret_cast<float4*>(base + kNoallocCtlBytes);                     // plane o at 0, plane d at n (as dr_trace_rays lays them out)
  uint2* hits = reinterpret_cast<uint2*>(base + kNoallocCtlBytes + kNoallocQueueBytes);
  // The array still holds the last call's counters: the fetch counter must start at zero.  Queue and hit entries need no clearing:
  // k_pack_rays writes entries 0 .. n-1 of both planes and k_trace writes a hit record for each of them before k_unpack_hits reads it.
  CUDA_TRY(cudaMemsetAsync(ctl, 0, 8, s));
  const uint32_t g = (n + 255) / 256;
  k_pack_rays<<<g, 256, 0, s>>>(o, d, n, q, n, ctl);
  k_trace<false><<<sc->n_sm, kTraceBlock, sc->trace_smem, s>>>(sc->dev, q, n, ctl, ctl + 1, hits, nullptr);
  k_unpack_hits<<<g, 256, 0, s>>>(sc->dev, hits, n, t, prim);
  CUDA_TRY(cudaGetLastError());
  return DR_OK;   // asynchronous: nothing is freed, so there is nothing to wait for
}
