// Chain kernels: propose (a1, a2, a10), decide (a7, a8, a11 + block kill counts), scan / scatter (a9),
// bootstrap (a0), resolve (a12); the target evaluation between propose and decide (a3-a6) is dr_eval.cuh.
// One thread = one chain; chain state is structure-of-arrays: x and score as d/4 planes of
// float4[N], so every load/store below is a coalesced 128-bit access (the paper's array-of-structs stateBuffer
// is prior art, not the layout used here).
#pragma once
#include "dr_eval.cuh"
#include "dr_rng.cuh"

namespace dr {

constexpr int kBlock = 256;      // streaming kernels

struct Counters {
  unsigned long long tours, mutations, rays, mh_accepts, nonfinite, grad_states, lit_init;
  uint32_t kills_last, queue_len, iteration, no_tour_resolves;
  uint32_t wave_timeouts, pad3[3];
  float p_lambda, kappa0, lambda, pad2;
  double psum;
};

struct ChainParams {
  int method;            // dr_method
  int restore, grad;
  uint32_t N, d, planes;
  float stddev, half_s2, c_tilde, dt, m, large_step_prob, p_lambda_override;
  int rao_blackwell;     // f3: weight = 1 / (lambda + kappa)
  int a_mode;            // f4: antisymmetric pattern of the drift
  uint32_t rho_grid;     // f4: regeneration density on G x G film tiles (0: uniform)
  const float2* rho;     //     (probability, running sum) per tile, row-major
  uint64_t seed;
  uint32_t epoch;
  uint32_t chain_offset;  // global id of chain 0 (RNG keying)
};

struct ChainState {
  // current state (rng field replaced by counter-based keying)
  float4* x;        // planes * N
  float4* g;        // planes * N, cached score of x (gradient methods)
  float4* fp;       // N: (f/p_hat rgb, p)
  uint32_t* pix;    // N
  uint32_t* sig;    // N
  uint8_t* killed;  // N
  // proposal
  float4* y;        // planes * N
  float4* gy;       // planes * N
  float4* fy;       // N: (f rgb, p)
  uint32_t* pixy;
  uint32_t* sigy;
  uint8_t* kind;    // 0 local move, 1 regeneration, 2 large step
  // last-step record + scheduling
  uint8_t* accepted;
  float* weight;
  uint32_t* order;  // evaluation order: alive chains ascending, then the regeneration queue ascending
  uint32_t* blockcnt;
  uint32_t* blockoff;
  double* partial;
  Counters* ctr;
};

__device__ __forceinline__ float wrap01(float v) {
  const float w = v - floorf(v);
  return fminf(w, 0x1.fffffep-1f);  // DESIGN.md Q3
}

// f4: x ~ rho from a uniform point -- the tile by inversion of the running sums with u0, uniform inside the tile (Q24)
__device__ __forceinline__ void regeneration_point(const ChainParams& cp, float& x0, float& x1) {
  const uint32_t G = cp.rho_grid, n = G * G;
  uint32_t lo = 0, hi = n - 1;                 // first tile t with x0 < cdf[t], else the last one
  while (lo < hi) {
    const uint32_t mid = (lo + hi) >> 1;
    if (x0 < __ldg(&cp.rho[mid]).y) hi = mid; else lo = mid + 1;
  }
  const float before = lo ? __ldg(&cp.rho[lo - 1]).y : 0.f;
  const float frac = (x0 - before) / __ldg(&cp.rho[lo]).x;
  x0 = wrap01(((float)(lo % G) + frac) / (float)G);
  x1 = wrap01(((float)(lo / G) + x1) / (float)G);
}
__device__ __forceinline__ float rho_at(const ChainParams& cp, float x0, float x1) {   // rho / rho_lambda
  const uint32_t G = cp.rho_grid;
  if (!G) return 1.0f;
  const uint32_t tx = min((uint32_t)floorf(x0 * (float)G), G - 1u), ty = min((uint32_t)floorf(x1 * (float)G), G - 1u);
  return (float)G * (float)G * __ldg(&cp.rho[ty * G + tx]).x;
}

__device__ __forceinline__ float4 mask_dims(float4 v, uint32_t plane, uint32_t d) {
  const uint32_t b = 4u * plane;
  if (b + 1 >= d) v.y = 0.f;
  if (b + 2 >= d) v.z = 0.f;
  if (b + 3 >= d) v.w = 0.f;
  return v;
}

// a1 + a2 + a10: build the proposal y of every chain for iteration n.
__global__ void __launch_bounds__(kBlock) k_propose(ChainParams cp, ChainState st, uint32_t n, int init) {
  const uint32_t i = blockIdx.x * kBlock + threadIdx.x;
  if (i >= cp.N) return;
  uint32_t kind = 0;
  if (init || (cp.restore && st.killed[i]) || cp.method == 5) kind = 1;   // path tracing: a fresh sample every iteration
  else if (!cp.restore) {
    const uint4 w = stream_block(cp.seed, cp.chain_offset + i, n, 0, P_DECIDE, cp.epoch);
    if (u01_co(w.x) < cp.large_step_prob) kind = 2;
  }
  st.kind[i] = (uint8_t)kind;
  const float s = cp.stddev, h = cp.half_s2, ct = cp.c_tilde;
  for (uint32_t j = 0; j < cp.planes; ++j) {
    const size_t at = (size_t)j * cp.N + i;
    float4 y;
    if (kind) {
      y = uniforms4(stream_block(cp.seed, cp.chain_offset + i, n, j, kind == 1 ? P_REGEN_U : P_LARGE_U, cp.epoch));
      if (j == 0 && kind == 1 && cp.rho_grid && (init || cp.restore)) regeneration_point(cp, y.x, y.y);   // x ~ nu = rho (Alg. 1, Alg. 2)
    } else {
      const float4 xi = normals4(stream_block(cp.seed, cp.chain_offset + i, n, j, P_PROP_N, cp.epoch));
      const float4 x = st.x[at];
      if (cp.method == 4 && cp.a_mode == 1 && 4 * j + 3 < cp.d) {   // f4: the two 2-blocks of the plane rotate into each other
        const float4 g = st.g[at];
        y.x = wrap01(((x.x + h * g.x) + ct * g.z) + s * xi.x);
        y.y = wrap01(((x.y + h * g.y) + ct * g.w) + s * xi.y);
        y.z = wrap01(((x.z + h * g.z) - ct * g.x) + s * xi.z);
        y.w = wrap01(((x.w + h * g.w) - ct * g.y) + s * xi.w);
      } else if (cp.method == 4) {  // Alg. 4: x += (s^2/2) g + c~ (g2, -g1) + s xi, per 2-block
        const float4 g = st.g[at];
        y.x = wrap01(((x.x + h * g.x) + ct * g.y) + s * xi.x);
        y.y = wrap01(((x.y + h * g.y) - ct * g.x) + s * xi.y);
        y.z = wrap01(((x.z + h * g.z) + ct * g.w) + s * xi.z);
        y.w = wrap01(((x.w + h * g.w) - ct * g.z) + s * xi.w);
      } else if (cp.grad) {  // MALA
        const float4 g = st.g[at];
        y.x = wrap01((x.x + h * g.x) + s * xi.x);
        y.y = wrap01((x.y + h * g.y) + s * xi.y);
        y.z = wrap01((x.z + h * g.z) + s * xi.z);
        y.w = wrap01((x.w + h * g.w) + s * xi.w);
      } else {  // Metropolis
        y.x = wrap01(x.x + s * xi.x);
        y.y = wrap01(x.y + s * xi.y);
        y.z = wrap01(x.z + s * xi.z);
        y.w = wrap01(x.w + s * xi.w);
      }
    }
    st.y[at] = mask_dims(y, j, cp.d);
    if (cp.grad) st.gy[at] = make_float4(0.f, 0.f, 0.f, 0.f);  // the evaluation writes only non-zero scores
  }
}

// a0: deterministic fp64 tree sum of p over the proposals of the init pass, then p_lambda, kappa0, lambda.
__global__ void __launch_bounds__(kBlock) k_psum_partial(ChainParams cp, ChainState st) {
  __shared__ double sm[kBlock];
  const uint32_t i = blockIdx.x * kBlock + threadIdx.x;
  double pi = 0.0;
  if (i < cp.N) {
    const float4 y0 = st.y[i];
    pi = (double)(st.fy[i].w / rho_at(cp, y0.x, y0.y));   // the init states are rho-distributed (f4); uniform rho: / 1
  }
  sm[threadIdx.x] = pi;
  __syncthreads();
  for (int s = kBlock / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sm[threadIdx.x] += sm[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) st.partial[blockIdx.x] = sm[0];
}

__global__ void __launch_bounds__(kBlock) k_bootstrap(ChainParams cp, ChainState st, uint32_t nblocks) {
  __shared__ double sm[kBlock];
  double acc = 0.0;
  for (uint32_t b = threadIdx.x; b < nblocks; b += kBlock) acc += st.partial[b];
  sm[threadIdx.x] = acc;
  __syncthreads();
  for (int s = kBlock / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sm[threadIdx.x] += sm[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    Counters* c = st.ctr;
    c->psum = sm[0];
    const float p_lambda = cp.p_lambda_override > 0.f ? cp.p_lambda_override : (float)(sm[0] / (double)cp.N + 1e-8);
    const float dt_eff = cp.method == 4 ? cp.dt : 1.0f;   // lambda == 1 for Metropolis-/MALA-Restore
    c->p_lambda = p_lambda;
    c->lambda = 1.0f / dt_eff;                              // L659
    c->kappa0 = p_lambda / (cp.m * dt_eff);                 // L752
  }
}

__device__ __forceinline__ float log_q_plane(float acc, float4 a, float4 ga, float4 b, float h) {   // acc += |delta|^2, coordinate by coordinate
  const float d0 = min_image(b.x - a.x - h * ga.x), d1 = min_image(b.y - a.y - h * ga.y);
  const float d2 = min_image(b.z - a.z - h * ga.z), d3 = min_image(b.w - a.w - h * ga.w);
  return (((acc + d0 * d0) + d1 * d1) + d2 * d2) + d3 * d3;
}

// a11: warp-aggregated vector atomic.  Lanes that splat to the same pixel are summed first, then one
// red.global.add.v4.f32 per distinct pixel.
__device__ __forceinline__ void splat(float4* accum, bool on, uint32_t pix, float4 v) {
  const unsigned active = __ballot_sync(0xFFFFFFFFu, on);
  if (!on) return;
  const unsigned lane = threadIdx.x & 31u;
  const unsigned peers = __match_any_sync(active, pix);
  const unsigned leader = __ffs(peers) - 1u;
  unsigned rem = lane == leader ? (peers & ~(1u << leader)) : 0u;
  const int rounds = __reduce_max_sync(active, __popc(peers) - 1);
  for (int r = 0; r < rounds; ++r) {
    const int src = rem ? __ffs(rem) - 1 : (int)lane;
    const float ax = __shfl_sync(active, v.x, src), ay = __shfl_sync(active, v.y, src);
    const float az = __shfl_sync(active, v.z, src), aw = __shfl_sync(active, v.w, src);
    if (rem) { v.x += ax; v.y += ay; v.z += az; v.w += aw; rem &= rem - 1u; }
  }
  if (lane == leader) atomicAdd(&accum[pix], v);
}

// a7 + a8 + a11 (+ per-block kill counts for a9).
__global__ void __launch_bounds__(kBlock) k_decide(ChainParams cp, ChainState st, float4* accum, uint32_t n, const uint32_t* wave_ctl) {
  const uint32_t i = blockIdx.x * kBlock + threadIdx.x;
  const bool in = i < cp.N;
  const Counters* c = st.ctr;
  bool killed = false, accepted_mh = false, do_splat = false, lit0 = false;
  uint32_t pix = 0;
  float4 contrib = make_float4(0.f, 0.f, 0.f, 0.f);
  if (in) {
    const uint4 w = stream_block(cp.seed, cp.chain_offset + i, n, 0, P_DECIDE, cp.epoch);
    const uint32_t kind = st.kind[i];
    const float4 fy = st.fy[i];
    lit0 = n == 0 && fy.w > 0.f;   // init pass: uniform samples with a contribution (zeta of SURVEY.md 8d)
    float4 cur = st.fp[i];
    pix = st.pix[i];
    bool take = true;
    if (kind != 1u && cp.method != 4) {  // Metropolis-Hastings test (not for regeneration / Langevin moves)
      const float px = cur.w + kEps, py = fy.w + kEps;
      float a = py / px;
      if (kind == 0u && cp.grad) {  // MALA: q(y->x) / q(x->y), minimal-image Gaussians (Q11)
        float fwd = 0.f, bwd = 0.f;
        for (uint32_t j = 0; j < cp.planes; ++j) {
          const size_t at = (size_t)j * cp.N + i;
          const float4 x = st.x[at], y = st.y[at], gx = st.g[at], gy = st.gy[at];
          bwd = log_q_plane(bwd, y, gy, x, cp.half_s2);
          fwd = log_q_plane(fwd, x, gx, y, cp.half_s2);
        }
        const float den = 2.0f * cp.stddev * cp.stddev;
        a *= expf((-bwd / den) - (-fwd / den));
      }
      if (!(a < 1.0f)) a = 1.0f;
      take = u01_co(w.y) < a;
      accepted_mh = take;
    }
    if (take) {
      for (uint32_t j = 0; j < cp.planes; ++j) {
        const size_t at = (size_t)j * cp.N + i;
        st.x[at] = st.y[at];
        if (cp.grad) st.g[at] = st.gy[at];
      }
      const float ph = fy.w + kEps;
      cur = make_float4(fy.x / ph, fy.y / ph, fy.z / ph, fy.w);   // f / p_hat (Alg. 1, Q9)
      if (cp.method == 5) cur = fy;                               // path tracing accumulates f itself
      pix = st.pixy[i];
      st.fp[i] = cur;
      st.pix[i] = pix;
      st.sig[i] = st.sigy[i];
    }
    // Accumulate (Alg. 1)
    const float phat = cur.w + kEps;
    float wgt = 1.0f;
    if (cp.restore) {
      float rho = 1.0f;
      if (cp.rho_grid) { const float4 x0 = st.x[i]; rho = rho_at(cp, x0.x, x0.y); }
      const float kappa = rho * c->kappa0 / phat;             // L445: (rho / rho_lambda) kappa0 / p_hat
      const float dt1 = -logf(u01_oc(w.z)) / c->lambda;       // L511
      const float dt2 = -logf(u01_oc(w.w)) / kappa;           // L512
      killed = !(dt1 < dt2);                                  // L513 (tie -> killed)
      wgt = killed ? dt2 : dt1;
      if (cp.rao_blackwell) wgt = 1.0f / (c->lambda + kappa);  // E[min(dt1, dt2)] (f3); the decision stays the race
      st.killed[i] = killed ? 1 : 0;
    }
    st.accepted[i] = take ? 1 : 0;
    st.weight[i] = wgt;
    do_splat = cur.w > 0.f;                                   // L522
    contrib = make_float4(wgt * cur.x, wgt * cur.y, wgt * cur.z, cp.method == 5 ? 1.0f : wgt / phat);  // L524 (+ ratio denominator, Q12; PT: count)
  }
  splat(accum, do_splat, pix, contrib);
  // block-level counts: kills (-> tourCount, regeneration queue) and MH accepts
  __shared__ uint32_t s_k, s_a, s_l;
  if (threadIdx.x == 0) { s_k = 0; s_a = 0; s_l = 0; }
  __syncthreads();
  const unsigned kb = __ballot_sync(0xFFFFFFFFu, killed), ab = __ballot_sync(0xFFFFFFFFu, accepted_mh), lb = __ballot_sync(0xFFFFFFFFu, lit0);
  if ((threadIdx.x & 31) == 0) {
    if (kb) atomicAdd(&s_k, (uint32_t)__popc(kb));
    if (ab) atomicAdd(&s_a, (uint32_t)__popc(ab));
    if (lb) atomicAdd(&s_l, (uint32_t)__popc(lb));
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    st.blockcnt[blockIdx.x] = s_k;
    if (s_k) atomicAdd(&st.ctr->tours, (unsigned long long)s_k);
    if (s_a) atomicAdd(&st.ctr->mh_accepts, (unsigned long long)s_a);
    if (s_l) atomicAdd(&st.ctr->lit_init, (unsigned long long)s_l);
    if (blockIdx.x == 0) {
      atomicAdd(&st.ctr->mutations, (unsigned long long)cp.N);
      st.ctr->iteration = n;
      if (wave_ctl && (wave_ctl[kCtlWaveError] & kErrTimeout)) st.ctr->wave_timeouts += 1;   // k_wave's watchdog fired in this iteration's evaluation (dr_wave.cuh)
    }
  }
}

// a9, step 2: exclusive scan of the per-block kill counts (one block; nblocks <= 16384 for N <= 2^22).
__global__ void __launch_bounds__(1024) k_scan(ChainState st, uint32_t nblocks) {
  __shared__ uint32_t sm[1024];
  const uint32_t per = (nblocks + 1023u) / 1024u;
  const uint32_t b0 = threadIdx.x * per;
  uint32_t sum = 0;
  for (uint32_t k = 0; k < per; ++k) if (b0 + k < nblocks) sum += st.blockcnt[b0 + k];
  sm[threadIdx.x] = sum;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {  // Hillis-Steele inclusive scan
    const uint32_t v = (int)threadIdx.x >= off ? sm[threadIdx.x - off] : 0u;
    __syncthreads();
    sm[threadIdx.x] += v;
    __syncthreads();
  }
  uint32_t run = sm[threadIdx.x] - sum;
  for (uint32_t k = 0; k < per; ++k)
    if (b0 + k < nblocks) { st.blockoff[b0 + k] = run; run += st.blockcnt[b0 + k]; }
  if (threadIdx.x == 1023) { st.ctr->queue_len = sm[1023]; st.ctr->kills_last = sm[1023]; }
}

// a9, step 3: stable scatter.  order[0 .. N-q) = alive chain ids ascending, order[N-q .. N) = killed ids
// ascending = the regeneration queue (Q13).  Warp ballot + popc prefix inside the block.
__global__ void __launch_bounds__(kBlock) k_scatter(ChainParams cp, ChainState st) {
  __shared__ uint32_t warp_off[kBlock / 32];
  const uint32_t i = blockIdx.x * kBlock + threadIdx.x;
  const bool k = i < cp.N && st.killed[i];
  const unsigned b = __ballot_sync(0xFFFFFFFFu, k);
  const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
  if (lane == 0) warp_off[wid] = __popc(b);
  __syncthreads();
  uint32_t before = 0;
  for (unsigned w = 0; w < wid; ++w) before += warp_off[w];
  before += __popc(b & ((1u << lane) - 1u));
  if (i < cp.N) {
    const uint32_t q = st.ctr->queue_len;
    const uint32_t kb = st.blockoff[blockIdx.x] + before;  // killed chains before i
    if (k) st.order[cp.N - q + kb] = i;
    else st.order[i - kb] = i;
  }
}

// a12: Alg. 3 with the pixel-count factor (Q2); plain MH: p_lambda / N_mut.  Totals: this shard's counters, or
// (sharded runs) externally reduced ones: ext_* != 0, or `tail` = the eight floats behind an all-reduced
// packed frame (k_pack_frame).
constexpr int kTailFloats = 8;
__device__ __forceinline__ unsigned long long limbs_to_u64(const float* t) {   // four sums of 16-bit limbs, each < 2^24: exact in fp32
  return (unsigned long long)t[0] + ((unsigned long long)t[1] << 16) + ((unsigned long long)t[2] << 32) + ((unsigned long long)t[3] << 48);
}
__global__ void __launch_bounds__(kBlock) k_resolve(ChainParams cp, Counters* c, const float4* accum, float* rgb,
                                                    uint32_t npix, unsigned long long ext_tours, unsigned long long ext_mut,
                                                    const float* tail) {
  const uint32_t q = blockIdx.x * kBlock + threadIdx.x;
  if (q >= npix) return;
  unsigned long long tours = c->tours, mut = c->mutations;
  if (tail) { tours = limbs_to_u64(tail); mut = limbs_to_u64(tail + 4); }
  else if (ext_mut) { tours = ext_tours; mut = ext_mut; }
  if (q == 0 && cp.restore && tours == 0) c->no_tour_resolves += 1;   // zero image, no division; reported by dr_chains_stats
  float scale;
  if (cp.restore) scale = tours ? (float)npix * c->kappa0 / (float)tours : 0.f;
  else if (cp.method == 5) scale = mut ? (float)npix / (float)mut : 0.f;
  else scale = mut ? (float)npix * c->p_lambda / (float)mut : 0.f;
  const float4 a = accum[q];
  rgb[3 * q] = scale * a.x; rgb[3 * q + 1] = scale * a.y; rgb[3 * q + 2] = scale * a.z;
}

// Sharded runs: one buffer per frame for ONE all-reduce(sum): the accumulation buffer followed by tourCount and the
// mutation count as 16-bit limbs in floats (sums over <= 256 ranks stay below 2^24, hence exact).
__global__ void __launch_bounds__(kBlock) k_pack_frame(const Counters* c, const float4* accum, float* buf, uint32_t npix) {
  const uint32_t q = blockIdx.x * kBlock + threadIdx.x;
  if (q < npix) reinterpret_cast<float4*>(buf)[q] = accum[q];
  if (q < (uint32_t)kTailFloats) {
    const unsigned long long v = q < 4 ? c->tours : c->mutations;
    buf[4 * (size_t)npix + q] = (float)((v >> (16 * (q & 3u))) & 0xFFFFull);
  }
}

// ---- Appendix C: bias field (L^* p_hat / p_hat) of the Alg. 4 dynamics on the 2-D analytic target ------
// b(y) = lambda (integral p(x) k(x, y) dx - p(y)) / p(y), lambda = 1 / dt, k = wrapped Gaussian of width s around
// m(x) = x + (s^2/2) g(x) + c~ (g2, -g1)(x).  Midpoint rule on M x M points; in double: the difference cancels to ~dt.
__device__ __forceinline__ void analytic_f64(const DevScene& sc, double x0, double x1, double& p, double& g0, double& g1) {
  double gx = 0.0, gy = 0.0;
  p = 0.0;
  for (int k = 0; k < sc.n_mix; ++k) {
    const double s = sc.mix_s[k], inv = 1.0 / s, norm = 0.3989422804014326779 * inv;
    double w[2], dw[2];
    const double dl[2] = {x0 - sc.mix_mx[k], x1 - sc.mix_my[k]};
    for (int a = 0; a < 2; ++a) {
      const double dm = dl[a] - floor(dl[a] + 0.5);
      w[a] = 0.0; dw[a] = 0.0;
      for (int j = -2; j <= 2; ++j) {
        const double z = (dm + (double)j) * inv, e = norm * exp(-0.5 * z * z);
        w[a] += e; dw[a] += -z * inv * e;
      }
    }
    p += sc.mix_w[k] * w[0] * w[1];
    gx += sc.mix_w[k] * dw[0] * w[1];
    gy += sc.mix_w[k] * w[0] * dw[1];
  }
  g0 = gx / (p + 1e-8);
  g1 = gy / (p + 1e-8);
}
__global__ void k_bias_table(DevScene sc, double s, double c_tilde, uint32_t M, double* tab) {   // tab: p | m0 | m1, M * M each
  const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= M * M) return;
  const double x0 = ((double)(k % M) + 0.5) / (double)M, x1 = ((double)(k / M) + 0.5) / (double)M;
  double p, g0, g1;
  analytic_f64(sc, x0, x1, p, g0, g1);
  const double h = 0.5 * s * s;
  tab[k] = p;
  tab[(size_t)M * M + k] = x0 + h * g0 + c_tilde * g1;
  tab[2 * (size_t)M * M + k] = x1 + h * g1 - c_tilde * g0;
}
__global__ void __launch_bounds__(256) k_bias_field(DevScene sc, double s, double dt, uint32_t G, uint32_t M, const double* tab, double* out) {
  __shared__ double sm[256];
  const uint32_t c = blockIdx.x;
  const double y0 = ((double)(c % G) + 0.5) / (double)G, y1 = ((double)(c / G) + 0.5) / (double)G;
  const double norm = 0.3989422804014326779 / s;
  const size_t MM = (size_t)M * M;
  double acc = 0.0;
  for (size_t k = threadIdx.x; k < MM; k += 256) {
    double d0 = y0 - tab[MM + k], d1 = y1 - tab[2 * MM + k];
    d0 -= floor(d0 + 0.5); d1 -= floor(d1 + 0.5);
    double w0 = 0.0, w1 = 0.0;
    for (int j = -1; j <= 1; ++j) {
      const double z0 = (d0 + (double)j) / s, z1 = (d1 + (double)j) / s;
      w0 += norm * exp(-0.5 * z0 * z0);
      w1 += norm * exp(-0.5 * z1 * z1);
    }
    acc += tab[k] * w0 * w1;
  }
  sm[threadIdx.x] = acc;
  __syncthreads();
  for (int st = 128; st > 0; st >>= 1) {
    if ((int)threadIdx.x < st) sm[threadIdx.x] += sm[threadIdx.x + st];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double p, g0, g1;
    analytic_f64(sc, y0, y1, p, g0, g1);
    out[c] = (1.0 / dt) * (sm[0] / (double)MM - p) / p;
  }
}

// ---- test hooks -------------------------------------------------------------------------------------------
// dr_trace_rays: user rays -> queue planes (o, d), and hits -> (t, original triangle id).
__global__ void k_pack_rays(const float* o, const float* d, uint32_t n, float4* q, uint32_t cap, uint32_t* cnt) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *cnt = n;
  if (i >= n) return;
  q[i] = make_float4(o[3 * i], o[3 * i + 1], o[3 * i + 2], 0.f);
  q[(size_t)cap + i] = make_float4(d[3 * i], d[3 * i + 1], d[3 * i + 2], 0.f);
}
__global__ void k_unpack_hits(DevScene sc, const uint2* hits, uint32_t n, float* t, uint32_t* prim) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint2 h = hits[i];
  if (h.y == kMiss) { t[i] = -1.f; prim[i] = 0xFFFFFFFFu; }
  else { t[i] = __uint_as_float(h.x); prim[i] = __float_as_uint(sc.tris[3 * h.y + 2].y); }
}

__global__ void k_philox_blocks(uint64_t seed, const uint32_t* ctr, uint32_t n, uint32_t* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 r = philox4x32_10(make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)),
                                make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]));
  out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

__global__ void k_rng_transforms(const uint32_t* words, uint32_t n, float* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float2 z = box_muller(words[2 * i], words[2 * i + 1]);
  out[4 * i] = u01_co(words[2 * i]); out[4 * i + 1] = u01_oc(words[2 * i]); out[4 * i + 2] = z.x; out[4 * i + 3] = z.y;
}

// SoA planes <-> row-major (download / upload hooks)
__global__ void k_planes_to_rows(const float4* planes, float* rows, uint32_t N, uint32_t d, uint32_t nplanes) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  for (uint32_t j = 0; j < nplanes; ++j) {
    const float4 q = planes[(size_t)j * N + i];
    const float v[4] = {q.x, q.y, q.z, q.w};
    for (uint32_t c = 0; c < 4 && 4 * j + c < d; ++c) rows[(size_t)i * d + 4 * j + c] = v[c];
  }
}
__global__ void k_rows_to_planes(const float* rows, float4* planes, uint32_t N, uint32_t d, uint32_t nplanes) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  for (uint32_t j = 0; j < nplanes; ++j) {
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    for (uint32_t c = 0; c < 4 && 4 * j + c < d; ++c) v[c] = rows[(size_t)i * d + 4 * j + c];
    planes[(size_t)j * N + i] = make_float4(v[0], v[1], v[2], v[3]);
  }
}
__global__ void k_fp_split(const float4* fp, float* p, float* fop, uint32_t N) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float4 q = fp[i];
  if (fop) { fop[3 * i] = q.x; fop[3 * i + 1] = q.y; fop[3 * i + 2] = q.z; }
  if (p) p[i] = q.w;
}
__global__ void k_fp_join(const float* p, const float* fop, float4* fp, uint32_t N) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  fp[i] = make_float4(fop[3 * i], fop[3 * i + 1], fop[3 * i + 2], p[i]);
}
__global__ void k_count_killed(ChainParams cp, ChainState st) {  // per-block kill counts after an upload
  __shared__ uint32_t s_k;
  if (threadIdx.x == 0) s_k = 0;
  __syncthreads();
  const uint32_t i = blockIdx.x * kBlock + threadIdx.x;
  const unsigned b = __ballot_sync(0xFFFFFFFFu, i < cp.N && st.killed[i]);
  if ((threadIdx.x & 31) == 0 && b) atomicAdd(&s_k, (uint32_t)__popc(b));
  __syncthreads();
  if (threadIdx.x == 0) st.blockcnt[blockIdx.x] = s_k;
}

}  // namespace dr
