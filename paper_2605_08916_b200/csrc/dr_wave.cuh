// k_wave: rows a3-a5 of one evaluation as ONE persistent kernel (the per-segment loop k_trace / k_shade of dr_eval.cuh
// computes the same results, state by state, and stays as the reference form and for the statistics pass).
//
// Why: a traversal launch ends with a tail in which its longest rays (about 100 dependent steps) keep every SM's
// block alive at falling occupancy; with 16 launches per frame that tail is a third of the traversal time
// (DESIGN.md section 6).  Here the rays of all segments go through one queue in global memory, so the queue only
// runs dry once, at the end of the evaluation:
//   * trace warps: the lockstep traversal of k_trace (trav_step); an idle lane takes the next ray of the queue.
//     A finished ray goes, as (state | segment, t, triangle), into a small ring in the block's shared memory.
//   * shade warps (kWaveShadeWarps<NEE, BLOCK> per block): take up to 32 finished rays from the block's ring, run shade_vertex
//     (the code of k_shade), write the surviving paths' next rays and count the finished paths.
// The evaluation is over when every path has finished (ctl[kCtlWaveDone] == n).
//
// Protocol (safe by construction, no timing assumption):
//   * A path has exactly one ray in flight.  The ray's data (origin, direction, throughput, signature: the three words
//     of a queue entry, dr_eval.cuh EvalWs) live in the 64-byte record of its STATE, so a record has one owner at a
//     time: the shade lane that writes it, then the trace lane that reads o, d, then the shade lane that reads all of
//     it and writes the next ray.  The hand-overs are the two below.
//   * The queue `ring` holds one 8-byte entry per ray, (state | (k - 1) << 27, tag), and is NEVER reused inside an
//     evaluation: it has L * cap entries and a path makes at most L rays.  Producers reserve indices with one atomic per
//     warp (ctl[kCtlWaveReserve]) and publish an entry with ONE 8-byte st.release after the record was written;
//     consumers claim kFetchChunk indices with one atomic (ctl[kCtlWaveHead]) and take an entry once its second word
//     equals this evaluation's tag (ws.tag, different for every evaluation that used the memory, 0 never: no clearing
//     between evaluations).  An entry is written once and read by one warp; indices past the last reservation are
//     never written and their claimants leave when the evaluation is over.
//   * The payload and its "ready" mark arrive in the same 8-byte word (no flag / data ordering on the reading side);
//     the record is then read at an address that depends on the payload, with __ldcg (L2, where the writer's release
//     made it visible); trace lane -> shade lane of the same block goes through shared memory (__threadfence_block).
//   Relaxed loads + __ldcg instead of ld.acquire / __threadfence(): on sm_100 those compile to CCTL.IVALL, which drops
//   the SM's whole L1 -- the L1 the traversal lives on (profiles/r01g_k_wave_full.md).
#pragma once
#include "dr_eval.cuh"

namespace dr {

#ifndef DR_WAVE_SHADE_WARPS
#define DR_WAVE_SHADE_WARPS 3
#endif
#ifndef DR_WAVE_SHADE_WARPS_NEE
#define DR_WAVE_SHADE_WARPS_NEE 5   // two visits per vertex and the emitter connection: 3 / 4 / 5 / 6 warps: 9.0 / 7.4 / 6.7 / 6.9 ms (r02f)
#endif
#ifndef DR_WAVE_REFILL_BELOW
#define DR_WAVE_REFILL_BELOW 26
#endif
#ifndef DR_WAVE_STALL_NS
#define DR_WAVE_STALL_NS 0      // test builds: every trace warp sleeps this long after each claim, before it reads the entries
#endif
#ifndef DR_CHECKS
#define DR_CHECKS 0             // test builds (compute-sanitizer is closed on this pool): device-side checks of the queue protocol;
#endif                          // a violated check sets a bit of ctl[kCtlWaveError], which the evaluation hooks turn into DR_ERR_CUDA
// kCtlWaveError and the kErr* bits are defined beside the other control words in dr_eval.cuh (k_decide reads the watchdog bit too)
#ifndef DR_WAVE_IDLE_LIMIT
#define DR_WAVE_IDLE_LIMIT (1u << 25)
#endif
#ifndef DR_WAVE_LOSE_RAY
#define DR_WAVE_LOSE_RAY 0      // test builds: the second rays of states 0..7 are never published, so the evaluation can only end by the watchdog
#endif
constexpr uint32_t kWaveIdleLimit = DR_WAVE_IDLE_LIMIT;   // idle rounds of >= 200 ns each (>= 6.7 s) before a trace warp gives up
#if DR_CHECKS
#define DR_CHECK(cond, bit) do { if (!(cond)) atomicOr(&ws.ctl[kCtlWaveError], (uint32_t)(bit)); } while (0)
#else
#define DR_CHECK(cond, bit) do { } while (0)
#endif
#ifndef DR_WAVE_SHADE_WARPS_NEE_SMALL
#define DR_WAVE_SHADE_WARPS_NEE_SMALL 3   // small evaluations do not keep five shade warps busy: 1.32 against 1.50 ms per frame at 2^14 chains
#endif
// shade warps of a block of BLOCK threads (the other warps trace)
template <bool NEE, int BLOCK> constexpr int kWaveShadeWarps =
    !NEE ? DR_WAVE_SHADE_WARPS : (BLOCK == TraceSmall::kBlock && TraceSmall::kBlock != TraceBig::kBlock ? DR_WAVE_SHADE_WARPS_NEE_SMALL : DR_WAVE_SHADE_WARPS_NEE);
constexpr int kWaveRefillBelow = DR_WAVE_REFILL_BELOW;   // a trace warp flushes its finished rays and refills below this many busy lanes
template <bool NEE, int BLOCK> constexpr int kWaveTraceThreads = BLOCK - 32 * kWaveShadeWarps<NEE, BLOCK>;
// evaluations of fewer states run in the small block shape (dr_eval.cuh TraceSmall); measured crossovers on configs[3]: between
// 2^18 and 589 824 states without, between 2^16 and 2^18 with next-event estimation (profiles/r02f_tuning.md)
constexpr uint32_t kWaveSmallBelow = 400000u, kWaveSmallBelowNee = 160000u;
// a chain ensemble knows better: the rays its last evaluation made (configs[3]: 3.6 M rays at 2^18 states are faster in the small
// shape, 8.2 M at 589 824 in the big one; with next-event estimation 2.6 M small, 5.2 M big; the caustic scene's 2.2 M rays at
// 2^20 states small: 0.97 against 1.16 ms)
constexpr uint32_t kWaveSmallBelowRays = 4500000u;
#ifndef DR_WAVE_HIT_CAP
#define DR_WAVE_HIT_CAP 1024
#endif
constexpr uint32_t kHitCap = DR_WAVE_HIT_CAP;   // entries of the block's ring of finished rays (power of two)
constexpr uint32_t kWaveKShift = 27; // payload = state | (k - 1) << 27 | shadow ray << 31
constexpr uint32_t kWaveStateMask = (1u << kWaveKShift) - 1u;


struct WaveShared {                  // counters of the block's ring (monotonic; index = counter & (kHitCap - 1))
  uint32_t reserve, pub, head, freed;
};
constexpr size_t kWaveExtraSmem = sizeof(WaveShared) + 3 * sizeof(uint32_t) * kHitCap;

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }

__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ uint2 ld_relaxed2(const uint2* p) {
  uint2 v;
  asm volatile("ld.relaxed.gpu.global.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release2(uint2* p, uint2 v) {
  asm volatile("st.release.gpu.global.v2.u32 [%0], {%1, %2};" ::"l"(p), "r"(v.x), "r"(v.y) : "memory");
}

// A trace warp with nothing to trace waits here until the entry it waits for (`next`) is published (returns 1; at once if its
// chunk is used up), every path has finished, or the watchdog fires (returns 2).  Not inlined: the wait must not cost the
// traversal loop registers.
__device__ __noinline__ uint32_t wave_idle_wait(const EvalWs& ws, uint32_t n, uint32_t next, bool chunk_done, uint32_t ring_cap) {
  const unsigned lane = threadIdx.x & 31u;
  for (uint32_t spins = 0;; ++spins) {
    uint32_t v = 0;
    if (lane == 0) {
      const bool ready = chunk_done || (next < ring_cap && ld_relaxed2(ws.ring + next).y == ws.tag);
      v = ld_relaxed(&ws.ctl[kCtlWaveDone]) >= n ? 2u : (ready ? 1u : 0u);
      if (!v && (spins & 0xFFFu) == 0xFFFu && (ld_relaxed(&ws.ctl[kCtlWaveError]) & kErrTimeout)) v = 2u;
      if (!v && spins > kWaveIdleLimit) { atomicOr(&ws.ctl[kCtlWaveError], (uint32_t)kErrTimeout); v = 2u; }
    }
    v = __shfl_sync(0xFFFFFFFFu, v, 0);
    if (v) return v;
    __nanosleep(200);
  }
}

// ---- the trace warps ------------------------------------------------------------------------------------------------
// NEE: shadow rays (payload bit 31) only ask whether the closest hit is the sampled emitter triangle.  They start with
// t_max just behind the sampled point and stop at the first other triangle hit clearly in front of it (kShadowBand): the
// closest hit is then not that emitter either way, so the visibility decision is the one of the full closest-hit query.
constexpr float kShadowBand = 1e-3f;
template <bool STATS, bool NEE, int BLOCK, int K>
__device__ __forceinline__ void wave_trace_loop(const DevScene& sc, const EvalWs& ws, uint32_t n, const uint4* smem, SmemStack<BLOCK>& st,
                                                SmemTriStack<BLOCK>& tst, WaveShared* wsh, uint32_t* h_pay, uint32_t* h_t, uint32_t* h_li,
                                                uint32_t one, unsigned long long* work) {
  const unsigned lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  constexpr unsigned kFull = 0xFFFFFFFFu;
  TravLane<K> L;
  uint32_t pay = 0, nn = 0, nt = 0;       // payload (state | segment) of the ray this lane holds
  trav_lane_init(L, one);
  uint32_t claim = 0, taken = kFetchChunk;  // the claimed chunk: entries claim + [taken, kFetchChunk) are still to be handed out
  uint32_t known = kFetchChunk;             // entries claim + [0, known) are known to be published
  uint32_t ent = 0;                         // lane j < kFetchChunk: payload of entry claim + j once it is known
  int poll = 0;
  bool pend = false;                        // this lane holds a finished ray that is not in the block's ring yet
  float sh_lim = -1.f;                      // NEE, shadow ray: an occluder closer than this ends the query (< 0: not a shadow ray)
  uint32_t sh_id = 0;                       //      the emitter triangle it aims at
  const uint32_t ring_cap = wave_ring_entries(sc, ws.cap);
  for (;;) {
    // ---- finished rays -> the block's ring (reserve, wait for room, write, publish in reservation order)
    {
      const unsigned dm = __ballot_sync(kFull, pend);
      if (dm) {
        const uint32_t cnt = __popc(dm);
        uint32_t base = 0;
        if (lane == 0) {
          base = atomicAdd(&wsh->reserve, cnt);
          while ((int)(base + cnt - ld_volatile(&wsh->freed)) > (int)kHitCap) __nanosleep(40);
          DR_CHECK(base + cnt - ld_volatile(&wsh->head) <= kHitCap, kErrHitRing);   // no unread entry is overwritten
        }
        base = __shfl_sync(kFull, base, 0);
        if (pend) {
          const uint32_t i = (base + __popc(dm & lt)) & (kHitCap - 1u);
          h_pay[i] = pay; h_t[i] = __float_as_uint(L.r.t); h_li[i] = L.r.li;
        }
        __syncwarp();
        if (lane == 0) {
          while (ld_volatile(&wsh->pub) != base) {}
          __threadfence_block();
          *reinterpret_cast<volatile uint32_t*>(&wsh->pub) = base + cnt;
        }
        __syncwarp();
        pend = false;
      }
    }
    // ---- hand rays to the idle lanes
    unsigned want = __ballot_sync(kFull, !L.active);
    while (want) {
      if (taken == kFetchChunk) {
        uint32_t b = 0;
        if (lane == 0) b = atomicAdd(&ws.ctl[kCtlWaveHead], kFetchChunk);
        claim = __shfl_sync(kFull, b, 0);
        taken = 0;
        known = 0;
        poll = 0;
#if DR_WAVE_STALL_NS > 0
        for (int z = 0; z < DR_WAVE_STALL_NS / 1000; ++z) __nanosleep(1000);
#endif
      }
      if (known < kFetchChunk && --poll <= 0) {  // which of the chunk's remaining entries are published?  (not asked every step)
        bool ok = false;
        if (lane >= known && lane < kFetchChunk && claim + lane < ring_cap) {
          const uint2 e = ld_relaxed2(ws.ring + claim + lane);
          ok = e.y == ws.tag;
          if (ok) ent = e.x;
        }
        const unsigned okm = __ballot_sync(kFull, ok) | ((1u << known) - 1u);
        known = min((uint32_t)__ffs(~okm) - 1u, kFetchChunk);   // length of the published prefix
        poll = 3;
      }
      if (known <= taken) break;  // nothing (more) of this chunk is published yet
      poll = 0;
      const uint32_t rank = __popc(want & lt);
      const bool mine = ((want >> lane) & 1u) && rank < known - taken;
      const uint32_t got_pay = __shfl_sync(kFull, ent, (taken + rank) & (kFetchChunk - 1u));
      if (mine) {
        pay = got_pay;
        const float4* e = ws.qa + kRecWords * (size_t)(pay & kWaveStateMask) + ((pay >> 31) ? 4u : 0u);   // the path's ray, or its shadow ray
        const float4 o = __ldcg(e), d = __ldcg(e + 1);   // written by another SM during this launch: not through L1
        DR_CHECK((pay & kWaveStateMask) < ws.cap && ((pay >> kWaveKShift) & 15u) < sc.L, kErrState);
        DR_CHECK((pay >> 31) || __float_as_uint(o.w) == (pay & kWaveStateMask), kErrOwner);   // the record is this state's
        trav_setup(L.r, o.x, o.y, o.z, d.x, d.y, d.z, one);
        trav_begin(L.s);
        L.tsp = 0;
        L.active = true;
        if (NEE) {
          sh_lim = -1.f;
          if (pay >> 31) { L.r.t = d.w * (1.0f + kShadowBand); sh_lim = d.w * (1.0f - kShadowBand); sh_id = __float_as_uint(o.w) & 0x0FFFFFFFu; }
        }
      }
      const unsigned got = __ballot_sync(kFull, mine);
      taken += __popc(got);
      want &= ~got;
    }
    unsigned act = __ballot_sync(kFull, L.active);
    if (!act) {  // nothing to trace: over, or waiting for the shade warps.  Spin here (counter local to this path) until the next
                 // claimed entry is published, every path has finished, or the watchdog gives up: the protocol cannot lose a
                 // path, but a kernel that never ends would take the GPU down with it.
      const bool over = wave_idle_wait(ws, n, claim + (taken == kFetchChunk ? kFetchChunk : known), taken == kFetchChunk, ring_cap) == 2u;
      if (over) break;
      poll = 0;
      continue;
    }
    // ---- lockstep traversal; a finished lane keeps its hit in L.r until the flush before the next refill
    do {
      bool done = trav_step<STATS, BLOCK, K>(sc, smem, st, tst, L, nn, nt);
      if (NEE && L.active && !done && sh_lim >= 0.f && L.r.id != 0xFFFFFFFFu && L.r.id != sh_id && L.r.t < sh_lim) {
        done = true;                                   // occluded: drop what is still requested or stacked
        L.has_node = false;
#pragma unroll
        for (int it = 0; it < K; ++it) L.tri[it].li = kMiss;
      }
      pend = pend || done;
      L.active = L.active && !done;
      act = __ballot_sync(kFull, L.active);
    } while (__popc(act) >= kWaveRefillBelow);
  }
  if (STATS) {   // the counting pass (dr_chains_work_stats, dr_eval_work_stats): node visits, triangle tests
    nn = __reduce_add_sync(kFull, nn);
    nt = __reduce_add_sync(kFull, nt);
    if (lane == 0) { atomicAdd(&work[0], (unsigned long long)nn); atomicAdd(&work[1], (unsigned long long)nt); }
  }
}

// ---- the shade warps ------------------------------------------------------------------------------------------------
template <bool GRAD, bool NEE>
__device__ __forceinline__ void wave_shade_loop(const DevScene& sc, const EvalWs& ws, const EvalIO& io, uint32_t n, WaveShared* wsh,
                                                const uint32_t* h_pay, const uint32_t* h_t, const uint32_t* h_li) {
  const unsigned lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  constexpr unsigned kFull = 0xFFFFFFFFu;
  const uint32_t ring_cap = wave_ring_entries(sc, ws.cap);
  for (;;) {
    // ---- take up to 32 finished rays of this block
    uint32_t head = 0, cnt = 0;
    if (lane == 0) {
      head = ld_volatile(&wsh->head);
      const uint32_t pub = ld_volatile(&wsh->pub);
      cnt = min(32u, pub - head);
      if (cnt && atomicCAS(&wsh->head, head, head + cnt) != head) cnt = 0xFFFFFFFFu;  // another shade warp was faster: again
    }
    head = __shfl_sync(kFull, head, 0);
    cnt = __shfl_sync(kFull, cnt, 0);
    if (cnt == 0xFFFFFFFFu) continue;
    if (cnt == 0) {
      uint32_t v = 0;
      if (lane == 0) v = ld_relaxed(&ws.ctl[kCtlWaveDone]) | (ld_relaxed(&ws.ctl[kCtlWaveError]) & kErrTimeout ? 0xFFFFFFFFu : 0u);
      if (__shfl_sync(kFull, v, 0) >= n) break;   // every path finished (or the watchdog fired)
      __nanosleep(100);
      continue;
    }
    __threadfence_block();
    const bool mine = lane < cnt;
    uint32_t pay = 0;
    uint2 h = make_uint2(0u, kMiss);
    if (mine) {
      const uint32_t i = (head + lane) & (kHitCap - 1u);
      pay = h_pay[i]; h.x = h_t[i]; h.y = h_li[i];
    }
    __syncwarp();
    if (lane == 0) {  // give the entries back, in order
      while (ld_volatile(&wsh->freed) != head) {}
      *reinterpret_cast<volatile uint32_t*>(&wsh->freed) = head + cnt;
    }
    // ---- shade.  With next-event estimation a vertex may take two visits: the hit of the path's ray (phase A: emitter
    // connection and direction sample; if the connection needs a shadow ray, that ray goes out first and the next ray
    // waits in the record), then the shadow ray's result (phase B, payload bit 31: visibility, signature, next ray).
    uint32_t bad = 0;
    const uint32_t s = pay & kWaveStateMask, k = ((pay >> kWaveKShift) & 15u) + 1u;
    const bool phase_b = (pay >> 31) != 0u;
    float4* rec = ws.qa + kRecWords * (size_t)s;
    bool want_grad = false, push = false;     // push: this lane publishes a queue entry (`entry`)
    uint32_t entry = 0;
    if (mine && !phase_b) {
      const float4 Q0 = __ldcg(rec), Q1 = __ldcg(rec + 1), Q2 = __ldcg(rec + 2);
      const float pb_prev = NEE ? __ldcg(rec + 3).w : -1.f;
      DR_CHECK(__float_as_uint(Q0.w) == s && k <= sc.L, kErrOwner);
#if DR_CHECKS
      if (!NEE) DR_CHECK(atomicAdd(&ws.hits[s].x, 1u) == k - 1u, kErrSegment);   // segments of a state are shaded once each, in order
#endif
      ShadeOut so;
      shade_vertex<GRAD, NEE>(sc, ws, io, k, Q0, Q1, Q2, pb_prev, h, s, so, bad);
      want_grad = so.want_grad;
      if (so.cont || so.shadow) {
        __stcg(rec, so.n0); __stcg(rec + 1, so.n1); __stcg(rec + 2, so.n2);
        if (NEE) __stcg(rec + 3, make_float4(so.cpend.x, so.cpend.y, so.cpend.z, so.pb_next));
        push = true;
        entry = s | (k << kWaveKShift);                       // the next ray: segment k + 1, stored as k
        if (NEE && so.shadow) {
          __stcg(rec + 4, make_float4(so.sh_o.x, so.sh_o.y, so.sh_o.z, __uint_as_float(so.light_id | (so.lobe << 28))));
          __stcg(rec + 5, make_float4(so.sh_d.x, so.sh_d.y, so.sh_d.z, so.sh_len));
          entry = s | ((k - 1u) << kWaveKShift) | 0x80000000u;   // the shadow ray of vertex k
        }
      }
    } else if (NEE && mine) {
      const float4 Q1 = __ldcg(rec + 1), Q2 = __ldcg(rec + 2), Q3 = __ldcg(rec + 3), S0 = __ldcg(rec + 4);
      if (io.nrays) __stcg(&io.nrays[s], __ldcg(&io.nrays[s]) + 1u);
      const uint32_t aim = __float_as_uint(S0.w);                      // emitter triangle | lobe << 28
      const bool vis = h.y != kMiss && __float_as_uint(__ldg(&sc.tris[3 * h.y + 2].y)) == (aim & 0x0FFFFFFFu);
      uint32_t info = __float_as_uint(Q2.w);
      if (vis) {
        float4 acc = __ldcg(&io.f[s]);
        acc.x += Q3.x; acc.y += Q3.y; acc.z += Q3.z;
        __stcg(&io.f[s], acc);
        info |= 1u << (16u + k);
      }
      const uint32_t sig = fnv(fnv(__float_as_uint(Q1.w), vis ? 7u : 6u), aim >> 28);
      if (Q2.x == 0.f && Q2.y == 0.f && Q2.z == 0.f) {         // the direction sample had zero weight: the path ends here
        finish_path<NEE>(sc, ws, io, k, s, 0.f, 0.f, 0.f, sig, info, k, kTermNone, GRAD, want_grad, bad);
      } else {
        __stcg(rec + 1, make_float4(Q1.x, Q1.y, Q1.z, __uint_as_float(sig)));
        __stcg(rec + 2, make_float4(Q2.x, Q2.y, Q2.z, __uint_as_float(info)));
        push = true;
        entry = s | (k << kWaveKShift);
      }
    }
    if (GRAD && !NEE) {  // reverse-pass list: one atomic per warp (with next-event estimation the sweep makes its own lists: dr_grad.cuh)
      const unsigned gm = __ballot_sync(kFull, want_grad);
      if (gm) {
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(&ws.ctl[kCtlGrad], (uint32_t)__popc(gm));
        base = __shfl_sync(kFull, base, 0);
        if (want_grad) ws.gradlist[base + __popc(gm & lt)] = s;
      }
    }
    // ---- the queue entries of the paths that go on (release: the records above are visible before the entry)
    const unsigned b = __ballot_sync(kFull, push);
    const uint32_t nc = __popc(b);
    if (nc) {
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(&ws.ctl[kCtlWaveReserve], nc);
      base = __shfl_sync(kFull, base, 0);
      DR_CHECK(base + nc <= ring_cap, kErrIndex);
#if DR_WAVE_LOSE_RAY
      if (push && s < 8u && k == 1u) push = false;   // reserved, never published
#endif
      if (push) st_release2(ws.ring + base + __popc(b & lt), make_uint2(entry, ws.tag));
    }
    if (lane == 0) {
      if (io.rays_ctr) atomicAdd(io.rays_ctr, (unsigned long long)cnt);
      if (cnt > nc) atomicAdd(&ws.ctl[kCtlWaveDone], cnt - nc);
    }
    if (io.nonfinite_ctr) {
      bad = __reduce_add_sync(kFull, bad);
      if (lane == 0 && bad) atomicAdd(io.nonfinite_ctr, (unsigned long long)bad);
    }
  }
}

// ---- the kernel -----------------------------------------------------------------------------------------------------
// NEE: the scene uses next-event estimation (two-phase vertices, shadow rays); STATS: the counting pass (NEE scenes only)
// C: the block shape, TraceBig or TraceSmall (dr_eval.cuh)
template <bool GRAD, bool STATS, bool NEE, class C>
__global__ void __launch_bounds__(C::kBlock, 1) k_wave(DevScene sc, EvalWs ws, EvalIO io, uint32_t n) {
  constexpr int kB = C::kBlock;
  static_assert((kFetchChunk & (kFetchChunk - 1u)) == 0 && kFetchChunk <= 32, "chunk: power of two, one entry per lane");
  extern __shared__ uint4 smem[];
  if (n == 0) return;
  // shared memory: one constant word | node stacks | triangle stacks | ring counters | ring
  SmemStack<kB> st{reinterpret_cast<uint2*>(smem + 1u) + threadIdx.x};
  SmemTriStack<kB> tst{st.base + (size_t)sc.stack_cap * kB, nullptr};
  tst.base3 = reinterpret_cast<uint32_t*>(tst.base + (size_t)kTriStack * kB - threadIdx.x) + threadIdx.x;
  uint32_t* tail = tst.base3 - threadIdx.x + (size_t)kTriStack * kB;
  WaveShared* wsh = reinterpret_cast<WaveShared*>(tail);
  uint32_t* h_pay = tail + sizeof(WaveShared) / 4;
  uint32_t* h_t = h_pay + kHitCap;
  uint32_t* h_li = h_t + kHitCap;
  if (threadIdx.x == 0) {
    smem[0].x = 0x3F800000u;
    wsh->reserve = 0; wsh->pub = 0; wsh->head = 0; wsh->freed = 0;
  }
  __syncthreads();
  const uint32_t one = *(volatile uint32_t*)&smem[0].x;  // dr_traverse.cuh qmagic
  if (threadIdx.x >= (unsigned)kWaveTraceThreads<NEE, kB>) wave_shade_loop<GRAD, NEE>(sc, ws, io, n, wsh, h_pay, h_t, h_li);
  else wave_trace_loop<STATS, NEE, kB, C::kTris>(sc, ws, n, smem, st, tst, wsh, h_pay, h_t, h_li, one, io.work);
}

}  // namespace dr
