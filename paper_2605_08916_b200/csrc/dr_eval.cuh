// Wavefront evaluation of the target for a batch of PSS states (rows a3-a6): x -> (f, p, pixel, score).
//   k_raygen            a3: camera ray of every state -> ray queue (state record + queue entry for k_wave)
//   rows a3-a5, two forms with identical results (dr_api.cu launch_eval):
//     k_wave (dr_wave.cuh)   ONE persistent kernel traces and shades all segments; the default
//     per segment k = 1..L:  k_trace  a4: persistent closest-hit kernel; a warp refills its idle lanes from the ray queue
//                            k_shade  a3/a5: shade_vertex for every ray of the segment; surviving paths are compacted
//                                     into the next queue (ballot + block-level prefix sum, one atomic per block)
//   k_grad              a6: reverse pass over the recorded vertices, only for the states that need it
//                       (with next-event estimation: k_grad_nee, dr_grad.cuh)
// shade_vertex (here) is one path vertex: emission / termination, emitter connection, direction sample; it calls
// vertex_fn<float> of dr_nee.cuh, the function the score kernels differentiate.  trav_step (here) is one lockstep step of
// the traversal, used by k_trace and k_wave.
// One thread = one ray / path vertex; nothing here is a dense contraction (no tensor cores).  The paper runs one
// shader thread per chain through a hardware ray-tracing pipeline; splitting the path into
// per-segment rays is what keeps 32-wide warps busy without RT cores (profiles/r01a: the one-thread-one-path
// kernel ran with 4.5 of 32 lanes active).
#pragma once
#include "dr_path.cuh"
#include "dr_nee.cuh"
#include "dr_traverse.cuh"

namespace dr {

#ifndef DR_STREAM_HINTS
#define DR_STREAM_HINTS 1   // evict-first stores of the vertex record, streaming loads of x in the shading: k_wave 4.33 -> 4.30 ms
#endif
#ifndef DR_TRACE_BLOCK
#define DR_TRACE_BLOCK 768   // 24 warps at 80 registers (with one triangle slot per lane): 640 / 704 / 768 / 896 / 1024 threads: profiles/r02f_tuning.md
#endif
#ifndef DR_TRI_STACK
#define DR_TRI_STACK 8
#endif
#ifndef DR_TRIS_PER_STEP
#define DR_TRIS_PER_STEP 1   // 2 slots: 11 more registers per thread (20 warps); 1 slot and 24 warps is 2.5 % faster (r02f)
#endif
#ifndef DR_REFILL_BELOW
#define DR_REFILL_BELOW 30
#endif
#ifndef DR_NODE_LD
#define DR_NODE_LD __ldg
#endif
#ifndef DR_TRI_LD
#define DR_TRI_LD __ldg
#endif
#ifndef DR_FETCH_CHUNK
#define DR_FETCH_CHUNK 32
#endif
constexpr int kTraceBlock = DR_TRACE_BLOCK;   // one persistent block per SM
constexpr int kTriStack = DR_TRI_STACK;      // postponed triangle groups per ray
constexpr int kTrisPerStep = DR_TRIS_PER_STEP;    // triangle tests per lockstep step
// The persistent traversal block comes in two shapes (profiles/r02f_tuning.md).  Big: 768 threads, one prefetched triangle per
// lane (80 registers): the most resident warps, best throughput, for evaluations that keep every lane supplied.  Small: 640
// threads, two triangle slots (96 registers): 12 % fewer lockstep steps per ray, for evaluations that wait on the latency of
// a path's dependent segments (below kWaveSmallBelow states: 25 % faster at 2^14 states, 8 % at 2^18).
#ifndef DR_TRACE_BLOCK_SMALL
#define DR_TRACE_BLOCK_SMALL 640
#endif
#ifndef DR_TRIS_PER_STEP_SMALL
#define DR_TRIS_PER_STEP_SMALL 2
#endif
struct TraceBig { static constexpr int kBlock = DR_TRACE_BLOCK, kTris = DR_TRIS_PER_STEP; };
struct TraceSmall { static constexpr int kBlock = DR_TRACE_BLOCK_SMALL, kTris = DR_TRIS_PER_STEP_SMALL; };
constexpr int kShadeBlock = 256;
constexpr int kGradBlock = 128;
constexpr uint32_t kFetchChunk = DR_FETCH_CHUNK;   // rays a warp takes from the queue per atomic
constexpr int kRefillBelow = DR_REFILL_BELOW;       // a warp goes back to the queue when fewer lanes than this hold a ray
constexpr uint32_t kSigInit = 2166136261u;
constexpr uint32_t kMiss = 0xFFFFFFFFu;

// control words of one evaluation (zeroed before k_raygen)
constexpr int kCtlCnt = 0;     // cnt[k], k = 1..L: rays of segment k
constexpr int kCtlHead = 20;   // head[k]: fetch counter of k_trace for segment k
constexpr int kCtlGrad = 40;   // states on the reverse-pass list
constexpr int kCtlGradKind = 64; // next-event estimation: entries of the reverse sweep's list (vertex index k, material kind) at [3 k + kind]
constexpr int kCtlWords = 128;

// Workspace for up to `cap` states.  Two forms of the same evaluation use it (same results, state by state):
//  * per-segment loop (k_trace / k_shade): ray queues qa, qb; an entry is three float4 in planes of `cap` entries,
//      Q0 = (o.xyz, bits(state)), Q1 = (d.xyz, bits(path signature)), Q2 = (T.rgb, bits(refract mask | has_ggx << 16));
//  * k_wave (dr_wave.cuh): the same three words live in a 96-byte record per STATE (kRecWords = 6 float4: qa[kRecWords s + 0..2],
//      words 3..5 carry the pending emitter connection and the shadow ray of next-event estimation; the memory of qa | qb),
//      and `ring` holds one 8-byte entry per ray: (state | (k - 1) << 27, tag of this evaluation).
struct EvalWs {
  float4* qa;          // 3 * cap; qb = qa + 3 * cap (one allocation of 6 * cap float4: k_wave uses all kRecWords * cap of it as records)
  float4* qb;          // 3 * cap
  uint2* hits;         // cap: (bits(t), triangle in leaf order or kMiss)   (loop form)
  uint2* ring;         // wave_ring_entries() ray entries, written once per evaluation, never reused      (k_wave)
  float4* rec;         // L * cap (score only): incoming direction and triangle of vertex k of state s at [k * cap + s]
                       //   next-event estimation: cap entries, the header of a finished path (masks, segments, terminal triangle, vertices)
  float4* vrec;        // next-event estimation + score: 3 * L * cap, the 48-byte record of the ray that reached vertex k = 1 .. L of
                       //   state s at [3 ((k - 1) cap + s)]: (direction, triangle | material kind << 30) (origin, density of the
                       //   direction) (throughput before the vertex, material index); the terminal emitter hit of a path is recorded too
  float4* adj;         // next-event estimation + score: 3 * cap, the 48-byte adjoint record of state s between the launches of
                       //   the reverse sweep at [3 s] (dr_grad.cuh)
  uint32_t* pinfo;     // cap (score only, else null): refract mask | rays << 16 of the finished path; with next-event estimation: the
                       //   material kinds of the path's vertices, two bits each (vertex k at bits 2 (k - 1)), OR-ed in by the shading
  uint32_t* gradlist;  // cap (score only); 3 * L * cap with next-event estimation: list (vertex index k, material kind) at [(3 k + kind) * cap, ...)
  uint32_t* ctl;       // kCtlWords
  uint32_t cap;
  uint32_t tag;        // k_wave: tag of this evaluation, != 0; ring entries of earlier evaluations carry other tags
};

// Inputs and outputs of one evaluation, all indexed by state s (planes: [plane * stride + s]).
struct EvalIO {
  const float4* x;       // PSS coordinates, d/4 planes
  size_t stride;
  const uint32_t* order; // optional: queue slot t evaluates state order[t]
  float4* g;             // score planes (score only); must be zero on entry
  float4* f;             // (f.rgb, p)
  uint32_t* pix;
  uint32_t* sig;
  uint32_t* nrays;       // optional
  unsigned long long* rays_ctr;       // optional: += closest-hit queries
  unsigned long long* nonfinite_ctr;  // optional: += states with non-finite f or score (Q18)
  unsigned long long* work;           // optional (k_trace<true>): work[0] += node visits, work[1] += triangle tests
  unsigned long long* grad_ctr;       // optional: += states that ran the reverse pass (k_grad)
};

__device__ __forceinline__ float2 x_pair(const EvalIO& io, uint32_t s, uint32_t k) {  // coordinates (2k, 2k+1)
#if DR_STREAM_HINTS
  const float4 q = __ldcs(&io.x[(size_t)(k >> 1) * io.stride + s]);
#else
  const float4 q = io.x[(size_t)(k >> 1) * io.stride + s];
#endif
  return (k & 1u) ? make_float2(q.z, q.w) : make_float2(q.x, q.y);
}
// the coordinates of vertex k: (u1, u2, v1, v2) = plane k with next-event estimation, else (u1, u2, 0, 0)
__device__ __forceinline__ float4 x_vertex(const DevScene& sc, const EvalIO& io, uint32_t s, uint32_t k) {
  if (sc.nee) return io.x[(size_t)k * io.stride + s];
  const float2 u = x_pair(io, s, k);
  return make_float4(u.x, u.y, 0.f, 0.f);
}
__device__ __forceinline__ void g_vertex(const DevScene& sc, const EvalIO& io, uint32_t s, uint32_t k, float4 g) {
  if (sc.nee) io.g[(size_t)k * io.stride + s] = g;
  else reinterpret_cast<float2*>(&io.g[(size_t)(k >> 1) * io.stride + s])[k & 1u] = make_float2(g.x, g.y);
}
__device__ __forceinline__ void g_pair(const EvalIO& io, uint32_t s, uint32_t k, float a, float b) {
  reinterpret_cast<float2*>(&io.g[(size_t)(k >> 1) * io.stride + s])[k & 1u] = make_float2(a, b);
}

// ---- a3: camera rays -------------------------------------------------------------------------------------------
// WAVE: the ray goes into the state's record and ring entry t (dr_wave.cuh); otherwise into slot t of queue qa.
constexpr int kCtlWaveReserve = 48, kCtlWaveHead = 50, kCtlWaveDone = 51;   // control words of k_wave
constexpr int kCtlWaveError = 52;   // k_wave: bits of the checks that fired (dr_wave.cuh); k_decide (dr_kernels.cuh) counts kErrTimeout into dr_stats.wave_timeouts
enum : uint32_t { kErrIndex = 1u, kErrState = 2u, kErrOwner = 4u, kErrSegment = 8u, kErrHitRing = 16u, kErrCount = 32u, kErrTimeout = 64u };
constexpr uint32_t kRecWords = 6;    // float4 per state record of k_wave: ray (o | state, d | signature, T | masks),
                                     // (pending emitter connection | density of the ray's direction), shadow ray (o | emitter id, lobe << 28; d | distance to the sampled point)
// queue entries an evaluation can need: a path makes at most L rays, and with next-event estimation one shadow ray per vertex
__host__ __device__ inline size_t wave_ring_entries(const DevScene& sc, size_t cap) { return (sc.nee ? 2u * sc.L - 1u : sc.L) * cap; }
template <bool WAVE>
__global__ void __launch_bounds__(kShadeBlock) k_raygen(DevScene sc, EvalWs ws, EvalIO io, uint32_t n) {
  const uint32_t t = blockIdx.x * kShadeBlock + threadIdx.x;
  if (t == 0) ws.ctl[WAVE ? kCtlWaveReserve : kCtlCnt + 1] = n;
  if (t >= n) return;
  const uint32_t s = io.order ? io.order[t] : t;
  const float4 x = io.x[s];
  io.pix[s] = pixel_of(x.x, x.y, sc.W, sc.H);
  const V3<float> d = camera_dir<float>(sc, x.x, x.y);
  const float4 q0 = make_float4(sc.cam_pos[0], sc.cam_pos[1], sc.cam_pos[2], __uint_as_float(s));
  const float4 q1 = make_float4(d.x, d.y, d.z, __uint_as_float(kSigInit));
  const float4 q2 = make_float4(1.f, 1.f, 1.f, __uint_as_float(0u));
  if (WAVE) {
    float4* r = ws.qa + kRecWords * (size_t)s;
    r[0] = q0; r[1] = q1; r[2] = q2;
    if (sc.nee) {
      r[3] = make_float4(0.f, 0.f, 0.f, -1.f);          // the camera ray has no direction density
      if (ws.pinfo) ws.pinfo[s] = 0u;                    // vertex kinds of this path (record_vertex)
      io.f[s] = make_float4(0.f, 0.f, 0.f, 0.f);        // emitter connections accumulate here
      if (io.nrays) io.nrays[s] = 0u;
    }
    ws.ring[t] = make_uint2(s, ws.tag);   // segment 1
  } else {
    ws.qa[t] = q0; ws.qa[(size_t)ws.cap + t] = q1; ws.qa[2 * (size_t)ws.cap + t] = q2;
  }
}

// ---- a4: closest hit, persistent ---------------------------------------------------------------------------------
// Per-thread stacks in shared memory, entry e of thread t at base[e * BLOCK] (bank = lane: conflict-free).
// Node groups grow up from entry 0; postponed triangle groups (tx, ty | tm) live in their own kTriStack entries above them.
template <int BLOCK> struct SmemStack {
  uint2* base;
  __device__ __forceinline__ void push(int sp, uint2 v) { base[sp * BLOCK] = v; }
  __device__ __forceinline__ uint2 pop(int sp) const { return base[sp * BLOCK]; }
};
template <int BLOCK> struct SmemTriStack {
  uint2* base;     // (tx, ty)
  uint32_t* base3; // tm
  __device__ __forceinline__ void push(int sp, const TravState& s) { base[sp * BLOCK] = make_uint2(s.tx, s.ty); base3[sp * BLOCK] = s.tm; }
  __device__ __forceinline__ void pop(int sp, TravState& s) const { const uint2 e = base[sp * BLOCK]; s.tx = e.x; s.ty = e.y; s.tm = base3[sp * BLOCK]; }
};

__device__ __forceinline__ void tri_one(const DevScene& sc, TravRay& r, TravState& s) {
  const uint32_t li = trav_next_tri(s);
  tri_test_bf(__ldg(&sc.tris[3 * li]), __ldg(&sc.tris[3 * li + 1]), __ldg(reinterpret_cast<const float2*>(&sc.tris[3 * li + 2])), li, true, r);
}

// One prefetched triangle of a lane: its three words are requested one step before they are tested.
struct TriSlot {
  float4 t0, t1;
  float2 t2;
  uint32_t li;  // leaf-order index, kMiss = empty
};

// One lockstep step of the traversal for this lane (parts A, N, T, F of the comment above k_trace).  Returns true if
// the lane's ray finished in this step (its closest hit is in r; the caller stores it and clears `active`).
template <int K> struct TravLane {
  TravRay r;
  TravState s;
  uint4 w0, w1, w2, w3, w4;      // words of the node to test next (valid if has_node)
  TriSlot tri[K];
  int tsp;                       // postponed triangle groups
  bool active, has_node;
};

template <int K> __device__ __forceinline__ void trav_lane_init(TravLane<K>& L, uint32_t one) {   // an idle lane
  L.active = false; L.has_node = false; L.tsp = 0;
  trav_setup(L.r, 0.f, 0.f, 0.f, 1.f, 1.f, 1.f, one);
  trav_begin(L.s);
  L.w0 = L.w1 = L.w2 = L.w3 = L.w4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
  for (int it = 0; it < K; ++it) { L.tri[it].li = kMiss; L.tri[it].t0 = L.tri[it].t1 = make_float4(0.f, 0.f, 0.f, 0.f); L.tri[it].t2 = make_float2(0.f, 0.f); }
}

template <bool STATS, int BLOCK, int K>
__device__ __forceinline__ bool trav_step(const DevScene& sc, const uint4* smem, SmemStack<BLOCK>& st, SmemTriStack<BLOCK>& tst, TravLane<K>& L,
                                          uint32_t& nn, uint32_t& nt) {
  TravRay& r = L.r;
  TravState& s = L.s;
  uint4 &w0 = L.w0, &w1 = L.w1, &w2 = L.w2, &w3 = L.w3, &w4 = L.w4;
  TriSlot* tri = L.tri;
  int& tsp = L.tsp;
  const bool active = L.active;
  bool& has_node = L.has_node;
  (void)smem;
  // The four parts are written without branches (selects and predicated loads / stores) so that the compiler can
  // interleave their dependency chains: with branches around every part each warp waited out the fixed latencies
  // of its bookkeeping one after the other (profiles/r01f_k_trace_full.md, step r01e: 53 % of the instructions took 78 % of the time).
  // A: node test
  {
    if (STATS) nn += has_node ? 1u : 0u;
    uint32_t h = node_hits(w0, w1, w2, w3, w4, r);
    h = has_node ? h : 0u;
    const uint32_t nty = h & 0x00FFFFFFu;
    const bool newtri = nty != 0u;
    bool keep_old = newtri && s.ty != 0u;  // triangles still pending from an earlier node: postpone them
    if (keep_old && tsp >= kTriStack) {    // (or test them now if their stack is full: rare)
      while (s.ty) { if (STATS) ++nt; tri_one(sc, r, s); }
      keep_old = false;
    }
    if (keep_old) tst.push(tsp, s);
    tsp += keep_old ? 1 : 0;
    s.tx = newtri ? w1.y : s.tx;
    s.ty = newtri ? nty : s.ty;
    s.tm = newtri ? w1.z : s.tm;
    s.gx = has_node ? w1.x : s.gx;
    s.gy = has_node ? ((h & 0xFF000000u) | w1.w) : s.gy;
  }
  // N: next node
  {
    const bool popn = active && !(s.gy & 0xFF000000u) && s.sp > 0;
    s.sp -= popn ? 1 : 0;
    if (popn) { const uint2 e = st.pop(s.sp); s.gx = e.x; s.gy = e.y; }
    const bool go = active && (s.gy & 0xFF000000u) != 0u;
    const uint32_t bit = top_bit(s.gy | 0x01000000u);
    const uint32_t rest = s.gy & ~(1u << bit);
    const bool keep = go && (rest & 0xFF000000u) != 0u;
    if (keep) st.push(s.sp, make_uint2(s.gx, rest));
    s.sp += keep ? 1 : 0;
    const uint32_t slot = (bit - 24u) ^ (r.octinv4 & 7u);
    const uint32_t node = s.gx + popc32(rest & ~(0xFFFFFFFFu << slot) & 0xFFu);
    s.gy = go ? rest : s.gy;
    if (go) {
      const uint4* np = sc.nodes + 5u * (size_t)node;
      w0 = DR_NODE_LD(np); w1 = DR_NODE_LD(np + 1); w2 = DR_NODE_LD(np + 2); w3 = DR_NODE_LD(np + 3); w4 = DR_NODE_LD(np + 4);
    }
    has_node = go;
  }
  // T: triangle tests
#pragma unroll
  for (int it = 0; it < K; ++it) {
    const bool valid = tri[it].li != kMiss;
    if (STATS) nt += valid ? 1u : 0u;
    tri_test_bf(tri[it].t0, tri[it].t1, tri[it].t2, tri[it].li, valid, r);  // reads every loaded word (dr_types.h TriPacked)
  }
  // F: next triangles
  {
    bool have_any = false;
#pragma unroll
    for (int it = 0; it < K; ++it) {
      const bool popt = active && s.ty == 0u && tsp > 0;
      tsp -= popt ? 1 : 0;
      if (popt) tst.pop(tsp, s);
      const bool have = active && s.ty != 0u;
      const uint32_t b = low_bit(s.ty | 0x80000000u);
      const uint32_t li = s.tx + popc32(s.tm & ~(0xFFFFFFFFu << b));
      s.ty = have ? (s.ty & (s.ty - 1u)) : s.ty;
      tri[it].li = have ? li : kMiss;
      if (have) {
        const float4* p = sc.tris + 3 * (size_t)li;
        tri[it].t0 = DR_TRI_LD(p); tri[it].t1 = DR_TRI_LD(p + 1); tri[it].t2 = DR_TRI_LD(reinterpret_cast<const float2*>(p + 2));
      }
      have_any = have_any || have;
    }
    return active && !(has_node || have_any);  // nothing requested, nothing pending: the ray is finished
  }
}

// q: planes Q0, Q1 of the queue (o, d).  Every warp takes kFetchChunk rays at a time from *head and keeps its lanes
// supplied from that private range.  The traversal runs in lockstep steps, software-pipelined one step deep so that
// every load has a phase of arithmetic between its issue and its first use (profiles/r01b: the un-pipelined loop
// spent 35 % of its warp-cycles waiting for the node and triangle words, one L2 round trip after the other):
//   A  node test of the node whose five words were requested in step k-1           (new children, new triangles)
//   N  choose the next node (nearest octant first), request its words               -> in flight during T
//   T  test the (up to kTrisPerStep) triangles whose words were requested in step k-1
//   F  choose the next triangles, request their words                               -> in flight during A of step k+1
// Lanes in different phases of different rays share the instructions of all four parts.
template <bool STATS>
__global__ void __launch_bounds__(kTraceBlock, 1)
k_trace(DevScene sc, const float4* __restrict__ q, uint32_t cap, const uint32_t* __restrict__ cnt, uint32_t* head,
        uint2* __restrict__ hits, unsigned long long* work) {
  extern __shared__ uint4 smem[];
  const uint32_t n = *cnt;
  if (n == 0) return;
  if (threadIdx.x == 0) smem[0].x = 0x3F800000u;   // one 16-byte word in front of the stacks
  __syncthreads();
  const uint32_t one = *(volatile uint32_t*)&smem[0].x;  // bits of 1.0f in a register the compiler cannot fold (dr_traverse.cuh qmagic)
  SmemStack<kTraceBlock> st{reinterpret_cast<uint2*>(smem + 1u) + threadIdx.x};
  SmemTriStack<kTraceBlock> tst{st.base + (size_t)sc.stack_cap * kTraceBlock, nullptr};
  tst.base3 = reinterpret_cast<uint32_t*>(tst.base + (size_t)kTriStack * kTraceBlock - threadIdx.x) + threadIdx.x;
  const unsigned lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  constexpr unsigned kFull = 0xFFFFFFFFu;
  uint32_t wnext = 0, wend = 0;  // this warp's private range of the queue
  bool drained = false;
  TravLane<kTrisPerStep> L;
  uint32_t ridx = 0, nn = 0, nt = 0;
  trav_lane_init(L, one);
  for (;;) {
    // ---- hand rays to the idle lanes
    unsigned want = __ballot_sync(kFull, !L.active);
    while (want && !drained) {
      if (wnext == wend) {
        uint32_t b = 0;
        if (lane == 0) b = atomicAdd(head, kFetchChunk);
        b = __shfl_sync(kFull, b, 0);
        if (b >= n) { drained = true; break; }
        wnext = b;
        wend = min(b + kFetchChunk, n);
      }
      const uint32_t rank = __popc(want & lt);
      const bool mine = ((want >> lane) & 1u) && rank < wend - wnext;
      if (mine) {
        ridx = wnext + rank;
        const float4 o = q[ridx], d = q[(size_t)cap + ridx];
        trav_setup(L.r, o.x, o.y, o.z, d.x, d.y, d.z, one);
        trav_begin(L.s);   // one work bit: the root, requested by part N of the first step
        L.tsp = 0;
        L.active = true;
      }
      const unsigned got = __ballot_sync(kFull, mine);
      wnext += __popc(got);
      want &= ~got;
    }
    unsigned act = __ballot_sync(kFull, L.active);
    if (!act) break;
    // ---- lockstep traversal
    do {
      const bool done = trav_step<STATS, kTraceBlock, kTrisPerStep>(sc, smem, st, tst, L, nn, nt);
      if (done) hits[ridx] = make_uint2(__float_as_uint(L.r.t), L.r.li);
      L.active = L.active && !done;
      act = __ballot_sync(kFull, L.active);
    } while (drained ? act != 0u : __popc(act) >= kRefillBelow);
  }
  if (STATS) {
    nn = __reduce_add_sync(kFull, nn);
    nt = __reduce_add_sync(kFull, nt);
    if (lane == 0) { atomicAdd(&work[0], (unsigned long long)nn); atomicAdd(&work[1], (unsigned long long)nt); }
  }
}

// Vertex k of one ray: emission / termination, emitter connection, direction sampling, throughput (rows a3 / a5).
// Q0..Q2 = the ray's words (dr_eval.cuh EvalWs), pb_prev = density of its direction (< 0: none, e.g. the camera ray or a
// Dirac lobe), h = (bits(t), triangle in leaf order or kMiss).  Three outcomes:
//   * the path ends here: f (added to what the emitter connections of earlier vertices left in io.f), p, signature are written;
//   * it continues (cont): the next ray is in n0..n2, the density of its direction in pb_next;
//   * with next-event estimation it may first need a shadow ray (shadow): sh_o / sh_d, the connection's contribution if it
//     is visible in cpend, the emitter triangle's id in light_id, and the lobe code still to be hashed into the signature
//     (n1.w then holds the signature BEFORE the visibility and the lobe); nee_finish() completes the vertex.
// Shared by k_shade (no next-event estimation) and k_wave.
struct ShadeOut {
  float4 n0, n1, n2;
  float pb_next;
  float3 sh_o, sh_d, cpend;
  float sh_len;          // distance from sh_o to the sampled emitter point
  uint32_t light_id, lobe;
  bool cont, shadow, want_grad;
};

constexpr uint32_t kTermNone = 0xFFFFFFFEu;   // the path ended without a terminal contribution (length cap, zero-weight direction)
// nv: vertices that sampled (1 .. nv), term: the triangle the last ray hit (leaf order), kMiss (environment) or kTermNone
template <bool NEE>
__device__ __forceinline__ void finish_path(const DevScene& sc_, const EvalWs& ws, const EvalIO& io, uint32_t k, uint32_t s, float f0, float f1,
                                            float f2, uint32_t sig, uint32_t info, uint32_t nv, uint32_t term, bool grad, bool& want_grad,
                                            uint32_t& bad) {
  const bool nee = NEE && sc_.nee;
  if (nee) { const float4 acc = __ldcg(&io.f[s]); f0 = acc.x + f0; f1 = acc.y + f1; f2 = acc.z + f2; }   // emitter connections so far
  float p = f0 * 0.2126f + f1 * 0.7152f + f2 * 0.0722f;
  if (!(isfinite(f0) && isfinite(f1) && isfinite(f2) && isfinite(p))) { f0 = f1 = f2 = p = 0.f; bad = 1; }
  __stcg(&io.f[s], make_float4(f0, f1, f2, p));
  io.sig[s] = sig;
  if (io.nrays && !nee) io.nrays[s] = k;
  if (grad) {
    if (nee) {
      ws.rec[s] = make_float4(__uint_as_float(info), __uint_as_float(k), __uint_as_float(term), __uint_as_float(nv));   // plane 0 of the vertex record
      want_grad = p > 0.f;                                                          // geometry and MIS terms depend on x
    } else {
      ws.pinfo[s] = (info & 0xFFFFu) | (k << 16);
      // only GGX weights depend on x: no GGX vertex or p == 0  =>  score == 0 exactly
      want_grad = (info >> 16) && p > 0.f;
    }
  }
}

// next-event estimation + score: what the reverse sweep (dr_grad.cuh) needs of the ray that reached vertex k
__device__ __forceinline__ size_t vrec_at(const EvalWs& ws, uint32_t k, uint32_t s) { return 3 * ((size_t)(k - 1u) * ws.cap + s); }
__device__ __forceinline__ void record_vertex(const EvalWs& ws, uint32_t k, uint32_t s, float3 o, float3 d, uint32_t li, uint32_t kind,
                                              uint32_t mi, float pb_prev, float T0, float T1, float T2) {
  float4* r = ws.vrec + vrec_at(ws, k, s);   // written once, read by the reverse sweep only: evict first
  __stcs(r, make_float4(d.x, d.y, d.z, __uint_as_float(li | (kind << 30))));
  __stcs(r + 1, make_float4(o.x, o.y, o.z, pb_prev));
  __stcs(r + 2, make_float4(T0, T1, T2, __uint_as_float(mi)));
  if (kind < 3u) atomicOr(&ws.pinfo[s], kind << (2u * (k - 1u)));   // no return value: a reduction at L2
}

template <bool GRAD, bool NEE>
__device__ __forceinline__ void shade_vertex(const DevScene& sc, const EvalWs& ws, const EvalIO& io, uint32_t k, const float4& Q0,
                                             const float4& Q1, const float4& Q2, float pb_prev, const uint2& h, uint32_t s, ShadeOut& out,
                                             uint32_t& bad) {
  const size_t cap = ws.cap;
  uint32_t sig = __float_as_uint(Q1.w), info = __float_as_uint(Q2.w);
  const float3 o = xyz(Q0), d = xyz(Q1);
  float T0 = Q2.x, T1 = Q2.y, T2 = Q2.z;
  float f0 = 0.f, f1 = 0.f, f2 = 0.f;
  bool done = true;
  uint32_t term = h.y;          // what the path's last ray hit, if it ends here with a contribution
  out.cont = false; out.shadow = false; out.want_grad = false;
  if (NEE && sc.nee && io.nrays) __stcg(&io.nrays[s], __ldcg(&io.nrays[s]) + 1u);   // L2: successive events of a path run on different SMs
  if (h.y == kMiss) {
    sig = fnv(sig, 0u);
    f0 = T0 * sc.env[0]; f1 = T1 * sc.env[1]; f2 = T2 * sc.env[2];
  } else {
    const uint32_t li = h.y;
    const float4 t0 = __ldg(&sc.tris[3 * li]), t1 = __ldg(&sc.tris[3 * li + 1]), t2 = __ldg(&sc.tris[3 * li + 2]);
    const float3 e1 = make_float3(t0.w, t1.x, t1.y), e2 = make_float3(t1.z, t1.w, t2.x);  // dr_types.h TriPacked
    sig = fnv(sig, __float_as_uint(t2.y) + 1u);
    const uint32_t mi = __float_as_uint(t2.z);
    const float4 m0 = __ldg(&sc.mats[3 * mi]), m1 = __ldg(&sc.mats[3 * mi + 1]);
    const uint32_t kind = __float_as_uint(m0.x);
    Frame fr;
    float dn;
    tri_frame(e1, e2, d, fr, dn);
    if (kind == 3u) {  // emitter: front face emits, path stops
      if (dn < 0.f) {
        sig = fnv(sig, 4u);
        const float4 m2 = __ldg(&sc.mats[3 * mi + 2]);
        const V3<float> ov{o.x, o.y, o.z}, dv{d.x, d.y, d.z};
        const float w_b = emitter_weight<float, NEE>(sc, xyz(t0), fr.nf, ov, dv, pb_prev, pb_prev >= 0.f);   // dn < 0: nf = n
        if (GRAD && NEE && sc.nee) record_vertex(ws, k, s, o, d, li, 3u, mi, pb_prev, T0, T1, T2);   // the reverse sweep starts here
        f0 = T0 * m1.z * w_b; f1 = T1 * m1.w * w_b; f2 = T2 * m2.x * w_b;
      } else {
        sig = fnv(sig, 5u);
        term = kTermNone;
      }
    } else if (k < sc.L) {
      term = kTermNone;
      const float4 u = x_vertex(sc, io, s, k);
      if (GRAD && NEE && sc.nee) record_vertex(ws, k, s, o, d, li, kind, mi, pb_prev, T0, T1, T2);
      else if (GRAD) __stcs(&ws.rec[(size_t)k * cap + s], make_float4(d.x, d.y, d.z, __uint_as_float(li)));   // written once, read by k_grad only: evict first
      const V3<float> ov{o.x, o.y, o.z}, dv{d.x, d.y, d.z};
      VertexOut<float> vo;
      V3<float> hit;
      bool reflect = false;
      uint32_t lj = 0;
      vertex_fn<float, NEE>(sc, xyz(t0), fr, dn, m0, m1, kind, ov, dv, u.x, u.y, u.z, u.w, true, reflect, vo, hit, lj);
      uint32_t lobe = kind == 0u ? 0u : (kind == 1u ? (reflect ? 1u : 2u) : 3u);
      if (kind == 1u && !reflect) info |= 1u << k;
      if (kind == 2u) info |= 1u << 16;
      T0 *= vo.W[0]; T1 *= vo.W[1]; T2 *= vo.W[2];
      const bool alive = !(T0 == 0.f && T1 == 0.f && T2 == 0.f);
      if (NEE && vo.nee_valid) {   // the vertex is completed by nee_finish() once the shadow ray is back
        const Light Lt = load_light(sc, lj);
        out.shadow = true;
        out.light_id = Lt.id;
        out.lobe = lobe;
        // (T fcos) (Le w_l / p_l): T here is the throughput BEFORE this vertex' direction sample
        out.cpend = make_float3((Q2.x * vo.fcos[0]) * vo.lw[0], (Q2.y * vo.fcos[1]) * vo.lw[1], (Q2.z * vo.fcos[2]) * vo.lw[2]);
        out.sh_o = make_float3(hit.x + fr.nf.x * sc.eps_ray, hit.y + fr.nf.y * sc.eps_ray, hit.z + fr.nf.z * sc.eps_ray);
        const float3 to_y = make_float3(vo.y.x, vo.y.y, vo.y.z) - out.sh_o;      // towards the sampled point, from the offset origin
        out.sh_len = sqrtf(dot3(to_y, to_y));
        out.sh_d = to_y * (1.0f / out.sh_len);                                    // == normalize3(to_y)
        done = false;
      } else {
        sig = fnv(sig, lobe);
      }
      if (alive || (NEE && vo.nee_valid)) {
        done = false;
        out.cont = alive && !(NEE && vo.nee_valid);
        out.n0 = make_float4(vo.o2.x, vo.o2.y, vo.o2.z, Q0.w);
        out.n1 = make_float4(vo.d2.x, vo.d2.y, vo.d2.z, __uint_as_float(sig));
        out.n2 = make_float4(T0, T1, T2, __uint_as_float(info));
        out.pb_next = vo.pb_valid ? vo.pb : -1.f;
      }
    } else {
      term = kTermNone;   // length cap on a surface: nothing is added
    }
  }
  if (done) finish_path<NEE>(sc, ws, io, k, s, f0, f1, f2, sig, info, k - 1u, term, GRAD, out.want_grad, bad);
}

// ---- a3 / a5: shade vertex k of every ray of segment k -------------------------------------------------------------
template <bool GRAD>
__global__ void __launch_bounds__(kShadeBlock) k_shade(DevScene sc, EvalWs ws, EvalIO io, uint32_t k) {   // scenes without next-event estimation
  __shared__ uint32_t s_warp[kShadeBlock / 32];
  __shared__ uint32_t s_base;
  const uint32_t n = ws.ctl[kCtlCnt + k];
  if (blockIdx.x * kShadeBlock >= n) return;  // whole block past the end of the queue
  const uint32_t j = blockIdx.x * kShadeBlock + threadIdx.x;
  const float4* qin = (k & 1u) ? ws.qa : ws.qb;
  float4* qout = (k & 1u) ? ws.qb : ws.qa;
  const size_t cap = ws.cap;
  ShadeOut so;
  so.cont = false; so.want_grad = false;
  uint32_t bad = 0, s = 0;
  if (j < n) {
    const float4 Q0 = qin[j], Q1 = qin[cap + j], Q2 = qin[2 * cap + j];
    s = __float_as_uint(Q0.w);
    shade_vertex<GRAD, false>(sc, ws, io, k, Q0, Q1, Q2, -1.f, ws.hits[j], s, so, bad);
  }
  const bool cont = so.cont, want_grad = so.want_grad;
  const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
  if (GRAD) {  // reverse-pass list: one atomic per warp
    const unsigned gm = __ballot_sync(0xFFFFFFFFu, want_grad);
    if (gm) {
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(&ws.ctl[kCtlGrad], (uint32_t)__popc(gm));
      base = __shfl_sync(0xFFFFFFFFu, base, 0);
      if (want_grad) ws.gradlist[base + __popc(gm & ((1u << lane) - 1u))] = s;
    }
  }
  // compaction of the surviving paths into the next queue: warp ballot, block prefix, one atomic per block
  const unsigned b = __ballot_sync(0xFFFFFFFFu, cont);
  if (lane == 0) s_warp[wid] = __popc(b);
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t tot = 0;
    for (int w = 0; w < kShadeBlock / 32; ++w) { const uint32_t c = s_warp[w]; s_warp[w] = tot; tot += c; }
    s_base = tot ? atomicAdd(&ws.ctl[kCtlCnt + k + 1], tot) : 0u;
    if (j == 0 && io.rays_ctr) atomicAdd(io.rays_ctr, (unsigned long long)n);
  }
  __syncthreads();
  if (cont) {
    const size_t at = s_base + s_warp[wid] + __popc(b & ((1u << lane) - 1u));
    qout[at] = so.n0; qout[cap + at] = so.n1; qout[2 * cap + at] = so.n2;
  }
  if (io.nonfinite_ctr) {
    bad = __reduce_add_sync(0xFFFFFFFFu, bad);
    if (lane == 0 && bad) atomicAdd(io.nonfinite_ctr, (unsigned long long)bad);
  }
}

// ---- a6: score by reverse accumulation -------------------------------------------------------------------------------
// With every discrete outcome frozen, grad p flows back from each GGX vertex through the chain of preceding specular
// vertices to the first diffuse vertex or the camera ("Score").  One thread = one listed state.
__global__ void __launch_bounds__(kGradBlock) k_grad(DevScene sc, EvalWs ws, EvalIO io) {
  const uint32_t idx = blockIdx.x * kGradBlock + threadIdx.x;
  if (idx == 0 && io.grad_ctr) atomicAdd(io.grad_ctr, (unsigned long long)ws.ctl[kCtlGrad]);
  if (idx >= ws.ctl[kCtlGrad]) return;
  const uint32_t s = ws.gradlist[idx];
  const size_t cap = ws.cap;
  const float4 fp = io.f[s];
  const uint32_t info = ws.pinfo[s];
  const uint32_t refract_mask = info & 0xFFFFu, nvert = (info >> 16) - 1u;  // vertices 1..nvert sampled a direction
  const float inv_phat = 1.0f / (fp.w + kEps);
  const float A0 = 0.2126f * fp.x, A1 = 0.7152f * fp.y, A2 = 0.0722f * fp.z;  // d p / d ln(w_c) per channel
  float db0 = 0.f, db1 = 0.f, db2 = 0.f;  // adjoint of the outgoing direction of the current vertex
  bool bad = false;
  for (uint32_t k = nvert; k >= 1; --k) {
    float ga = 0.f, gb = 0.f;
    const float4 rc = ws.rec[(size_t)k * cap + s];
    const uint32_t li = __float_as_uint(rc.w);
    const float3 din = xyz(rc);
    const float4 t0 = __ldg(&sc.tris[3 * li]), t1 = __ldg(&sc.tris[3 * li + 1]), t2 = __ldg(&sc.tris[3 * li + 2]);
    const float3 e1 = make_float3(t0.w, t1.x, t1.y), e2 = make_float3(t1.z, t1.w, t2.x);
    const uint32_t mi = __float_as_uint(t2.z);
    const float4 m0 = __ldg(&sc.mats[3 * mi]), m1 = __ldg(&sc.mats[3 * mi + 1]);
    const uint32_t kind = __float_as_uint(m0.x);
    Frame fr;
    float dn;
    tri_frame(e1, e2, din, fr, dn);
    const float2 u = x_pair(io, s, k);
    const bool live = db0 != 0.f || db1 != 0.f || db2 != 0.f;
    if (kind == 0u) {
      if (live) {
        const V3<Du<2>> w = lambert_dir<Du<2>>(fr, du_var<2>(u.x, 0), du_var<2>(u.y, 1));
        ga = db0 * w.x.d[0] + db1 * w.y.d[0] + db2 * w.z.d[0];
        gb = db0 * w.x.d[1] + db1 * w.y.d[1] + db2 * w.z.d[1];
      }
      db0 = db1 = db2 = 0.f;  // a diffuse vertex forgets the incoming direction
    } else if (kind == 1u) {
      if (live) {
        const float eta = dn < 0.f ? m1.x : 1.0f / m1.x;
        V3<Du<3>> di{du_var<3>(din.x, 0), du_var<3>(din.y, 1), du_var<3>(din.z, 2)};
        const V3<Du<3>> w = dielectric_dir<Du<3>>(fr, eta, !((refract_mask >> k) & 1u), di);
        const float n0 = db0 * w.x.d[0] + db1 * w.y.d[0] + db2 * w.z.d[0];
        const float n1 = db0 * w.x.d[1] + db1 * w.y.d[1] + db2 * w.z.d[1];
        const float n2 = db0 * w.x.d[2] + db1 * w.y.d[2] + db2 * w.z.d[2];
        db0 = n0; db1 = n1; db2 = n2;
      }
    } else if (kind == 2u) {
      V3<Du<5>> di{du_var<5>(din.x, 2), du_var<5>(din.y, 3), du_var<5>(din.z, 4)};
      V3<Du<5>> w;
      Du<5> c5, G1;
      if (ggx_dir<Du<5>>(fr, m1.y, di, du_var<5>(u.x, 0), du_var<5>(u.y, 1), w, c5, G1)) {
        // S = sum_c (A_c / w_c) w_c(x) with w_c = (F0_c + (1 - F0_c) c5) G1
        const float w0 = (m0.y + (1.0f - m0.y) * c5.v) * G1.v, w1 = (m0.z + (1.0f - m0.z) * c5.v) * G1.v,
                    w2 = (m0.w + (1.0f - m0.w) * c5.v) * G1.v;
        const float B0 = w0 > 0.f ? A0 / w0 : 0.f, B1 = w1 > 0.f ? A1 / w1 : 0.f, B2 = w2 > 0.f ? A2 / w2 : 0.f;
        const float a0 = B0 * m0.y + B1 * m0.z + B2 * m0.w;
        const float a1 = B0 * (1.0f - m0.y) + B1 * (1.0f - m0.z) + B2 * (1.0f - m0.w);
        const Du<5> S = G1 * (c5 * a1 + a0);
        float nj[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) nj[j] = db0 * w.x.d[j] + db1 * w.y.d[j] + db2 * w.z.d[j] + S.d[j];
        ga = nj[0]; gb = nj[1];
        db0 = nj[2]; db1 = nj[3]; db2 = nj[4];
      }
    }
    ga *= inv_phat; gb *= inv_phat;
    bad = bad || !(isfinite(ga) && isfinite(gb));
    g_pair(io, s, k, ga, gb);
  }
  {
    float ga = 0.f, gb = 0.f;
    if (db0 != 0.f || db1 != 0.f || db2 != 0.f) {
      const float4 x = io.x[s];
      const V3<Du<2>> w = camera_dir<Du<2>>(sc, du_var<2>(x.x, 0), du_var<2>(x.y, 1));
      ga = (db0 * w.x.d[0] + db1 * w.y.d[0] + db2 * w.z.d[0]) * inv_phat;
      gb = (db0 * w.x.d[1] + db1 * w.y.d[1] + db2 * w.z.d[1]) * inv_phat;
    }
    bad = bad || !(isfinite(ga) && isfinite(gb));
    g_pair(io, s, 0, ga, gb);
  }
  if (bad) {  // Q18: a non-finite score makes the state a zero-contribution state
    io.f[s] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (uint32_t k = 0; k <= nvert; ++k) g_pair(io, s, k, 0.f, 0.f);
    if (io.nonfinite_ctr) atomicAdd(io.nonfinite_ctr, 1ull);
  }
}

// ---- the 2-D analytic target (no rays) -----------------------------------------------------------------------------------
template <bool GRAD>
__global__ void __launch_bounds__(kShadeBlock) k_eval_analytic(DevScene sc, EvalIO io, uint32_t n) {
  const uint32_t t = blockIdx.x * kShadeBlock + threadIdx.x;
  if (t >= n) return;
  const uint32_t s = io.order ? io.order[t] : t;
  const float4 x = io.x[s];
  float p, g0, g1;
  eval_analytic(sc, x.x, x.y, p, g0, g1);
  const bool bad = !isfinite(p) || (GRAD && !(isfinite(g0) && isfinite(g1)));
  if (bad) { p = 0.f; g0 = g1 = 0.f; if (io.nonfinite_ctr) atomicAdd(io.nonfinite_ctr, 1ull); }
  io.f[s] = make_float4(p, p, p, p);
  io.pix[s] = pixel_of(x.x, x.y, sc.W, sc.H);
  io.sig[s] = 0u;
  if (io.nrays) io.nrays[s] = 0u;
  if (GRAD) g_pair(io, s, 0, g0, g1);
}

}  // namespace dr
