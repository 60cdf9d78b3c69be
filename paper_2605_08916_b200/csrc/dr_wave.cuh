// k_wave: rows a3-a5 of one evaluation as ONE persistent kernel (used for evaluations of at least kWaveMinStates
// states; smaller ones and the statistics pass use the per-segment loop k_trace / k_shade of dr_eval.cuh; same
// results, state by state).
//
// Why: a traversal launch ends with a tail in which its longest rays (about 100 dependent steps) keep every SM's
// block alive at falling occupancy; with 16 launches per frame that tail is a third of the traversal time
// (DESIGN.md section 6).  Here the rays of all segments go through one ring in global memory, so the queue only
// runs dry once, at the end of the evaluation:
//   * trace warps: the lockstep traversal of k_trace (trav_step); an idle lane takes the next ray from the ring.
//     A finished ray goes, as (slot, t, triangle), into a small ring in the block's shared memory.
//   * shade warps (kWaveShadeWarps per block): take up to 32 finished rays from the block's ring, run shade_vertex
//     (the code of k_shade), append the surviving paths' next rays to the global ring and count the finished paths.
// The evaluation is over when every path has finished (ctl[kCtlWaveDone] == n).
//
// Global ring: slot i of the ring is entry i mod 2 cap of (qa | qb) (dr_eval.cuh EvalWs), three planes per entry.
// Producers reserve with one atomic per warp (ctl[kCtlWaveReserve]), write the entry and then its ready word
// (ws.hits reused as uint32 ready[2 cap]: lap + 1 of the index that was written, release / acquire); consumers claim
// kFetchChunk slots with one atomic (ctl[kCtlWaveHead]) and take a slot once its ready word shows their lap.
// (A single "published up to" counter advanced in reservation order was measured first: it serialises all shade
// warps on one L2 round trip per batch, 35 M rays/s.)  A path has at most one ray in flight, slots are consumed in order, so a slot is never reused
// before it was read (capacity 2 cap >= 2 n).  The segment index k of a ray travels in the top five bits of Q0.w.
#pragma once
#include "dr_eval.cuh"

namespace dr {

#ifndef DR_WAVE_SHADE_WARPS
#define DR_WAVE_SHADE_WARPS 3
#endif
#ifndef DR_WAVE_REFILL_BELOW
#define DR_WAVE_REFILL_BELOW 26
#endif
constexpr int kWaveShadeWarps = DR_WAVE_SHADE_WARPS;     // sweep 1 / 2 / 3 / 4 / 5 / 6: 9.13 / 5.25 / 4.85 / 5.05 / 5.22 / 5.45 ms per frame
constexpr int kWaveRefillBelow = DR_WAVE_REFILL_BELOW;   // a trace warp flushes its finished rays and refills below this many busy lanes
constexpr int kWaveTraceThreads = kTraceBlock - 32 * kWaveShadeWarps;
constexpr uint32_t kHitCap = 1024;   // entries of the block's ring of finished rays (power of two)
constexpr int kCtlWaveReserve = 48, kCtlWaveHead = 50, kCtlWaveDone = 51;
constexpr uint32_t kWaveKShift = 27; // Q0.w = state | k << 27

struct WaveShared {                  // counters of the block's ring (monotonic; index = counter & (kHitCap - 1))
  uint32_t reserve, pub, head, freed;
};
constexpr size_t kWaveExtraSmem = sizeof(WaveShared) + 3 * sizeof(uint32_t) * kHitCap;

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }

__device__ __forceinline__ float4* ring_entry(const EvalWs& ws, uint32_t i) {
  const uint32_t j = i % (2u * ws.cap);
  return j < ws.cap ? ws.qa + j : ws.qb + (j - ws.cap);
}

// initial state of the ring after k_raygen wrote n camera rays into qa[0 .. n)
__global__ void k_wave_begin(EvalWs ws, uint32_t n) {   // ready[] was zeroed by the host
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t == 0) { ws.ctl[kCtlWaveReserve] = n; ws.ctl[kCtlWaveHead] = 0; ws.ctl[kCtlWaveDone] = 0; }
  if (t < n) reinterpret_cast<uint32_t*>(ws.hits)[t] = 1u;
}

// Flags and counters are read with a relaxed gpu-scope load (served by L2) and the data they guard with __ldcg, never
// with an acquire load or a gpu-scope fence: on sm_100 those end in CCTL.IVALL, which drops the whole L1 of the SM -- the
// L1 the traversal lives on (first version of this kernel: l1tex hit rate 53 -> 46 %, lts hit rate 88 -> 76 %).
// st.release is MEMBAR + store without the invalidation, so the writers keep it.
__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---- the trace warps ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void wave_trace_loop(const DevScene& sc, const EvalWs& ws, uint32_t n, const uint4* smem, SmemStack& st,
                                                SmemTriStack& tst, WaveShared* wsh, uint32_t* h_slot, uint32_t* h_t, uint32_t* h_li,
                                                uint32_t one) {
  const unsigned lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  constexpr unsigned kFull = 0xFFFFFFFFu;
  const size_t cap = ws.cap;
  TravLane L;
  uint32_t ridx = 0, nn = 0, nt = 0;
  L.active = false; L.has_node = false; L.tsp = 0;
  trav_setup(L.r, 0.f, 0.f, 0.f, 1.f, 1.f, 1.f, one);
  trav_begin(L.s);
  L.w0 = L.w1 = L.w2 = L.w3 = L.w4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
  for (int it = 0; it < kTrisPerStep; ++it) { L.tri[it].li = kMiss; L.tri[it].t0 = L.tri[it].t1 = make_float4(0.f, 0.f, 0.f, 0.f); L.tri[it].t2 = make_float2(0.f, 0.f); }
  uint32_t claim = 0, taken = kFetchChunk;  // the claimed chunk: ring slots claim + [taken, kFetchChunk) are still to be handed out
  uint32_t known = kFetchChunk;             // slots claim + [0, known) are known to be written
  int poll = 0;
  bool pend = false;                        // this lane holds a finished ray that is not in the block's ring yet
  uint32_t* ready = reinterpret_cast<uint32_t*>(ws.hits);
  const uint32_t ring = 2u * ws.cap;
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
        }
        base = __shfl_sync(kFull, base, 0);
        if (pend) {
          const uint32_t i = (base + __popc(dm & lt)) & (kHitCap - 1u);
          h_slot[i] = ridx; h_t[i] = __float_as_uint(L.r.t); h_li[i] = L.r.li;
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
      }
      if (known < kFetchChunk && --poll <= 0) {  // which of the chunk's remaining slots are written?  (not asked every step)
        bool ok = false;
        if (lane >= known && lane < kFetchChunk) {
          const uint32_t idx = claim + lane;
          ok = ld_relaxed(ready + idx % ring) == idx / ring + 1u;
        }
        const unsigned okm = __ballot_sync(kFull, ok) | ((1u << known) - 1u);
        known = min((uint32_t)__ffs(~okm) - 1u, kFetchChunk);   // length of the ready prefix
        __syncwarp();
        poll = 3;
      }
      const uint32_t avail = known;
      if (avail <= taken) break;  // nothing (more) of this chunk is written yet
      poll = 0;
      const uint32_t rank = __popc(want & lt);
      const bool mine = ((want >> lane) & 1u) && rank < avail - taken;
      if (mine) {
        ridx = claim + taken + rank;
        const float4* e = ring_entry(ws, ridx);
        const float4 o = __ldcg(e), d = __ldcg(e + cap);   // written by another SM during this launch: not through L1
        trav_setup(L.r, o.x, o.y, o.z, d.x, d.y, d.z, one);
        trav_begin(L.s);
        L.tsp = 0;
        L.active = true;
      }
      const unsigned got = __ballot_sync(kFull, mine);
      taken += __popc(got);
      want &= ~got;
    }
    unsigned act = __ballot_sync(kFull, L.active);
    if (!act) {  // nothing to trace: over, or waiting for the shade warps
      uint32_t v = 0;
      if (lane == 0) v = ld_relaxed(&ws.ctl[kCtlWaveDone]);
      if (__shfl_sync(kFull, v, 0) >= n) break;
      __nanosleep(200);
      poll = 0;
      continue;
    }
    // ---- lockstep traversal; a finished lane keeps its hit in L.r until the flush before the next refill
    do {
      const bool done = trav_step<false>(sc, smem, st, tst, L, nn, nt);
      pend = pend || done;
      L.active = L.active && !done;
      act = __ballot_sync(kFull, L.active);
    } while (__popc(act) >= kWaveRefillBelow);
  }
}

// ---- the shade warps ------------------------------------------------------------------------------------------------
template <bool GRAD>
__device__ __forceinline__ void wave_shade_loop(const DevScene& sc, const EvalWs& ws, const EvalIO& io, uint32_t n, WaveShared* wsh,
                                                const uint32_t* h_slot, const uint32_t* h_t, const uint32_t* h_li) {
  const unsigned lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
  constexpr unsigned kFull = 0xFFFFFFFFu;
  constexpr uint32_t kStateMask = (1u << kWaveKShift) - 1u;
  const size_t cap = ws.cap;
  for (;;) {
    // ---- take up to 32 finished rays of this block
    uint32_t head = 0, cnt = 0;
    if (lane == 0) {
      head = ld_volatile(&wsh->head);
      const uint32_t pub = ld_volatile(&wsh->pub);
      cnt = min(32u, pub - head);
      if (cnt && atomicCAS(&wsh->head, head, head + cnt) != head) cnt = 0xFFFFFFFFu;  // the other shade warp was faster: again
    }
    head = __shfl_sync(kFull, head, 0);
    cnt = __shfl_sync(kFull, cnt, 0);
    if (cnt == 0xFFFFFFFFu) continue;
    if (cnt == 0) {
      uint32_t v = 0;
      if (lane == 0) v = ld_relaxed(&ws.ctl[kCtlWaveDone]);
      if (__shfl_sync(kFull, v, 0) >= n) break;
      __nanosleep(100);
      continue;
    }
    __threadfence_block();
    const bool mine = lane < cnt;
    uint32_t slot = 0;
    uint2 h = make_uint2(0u, kMiss);
    if (mine) {
      const uint32_t i = (head + lane) & (kHitCap - 1u);
      slot = h_slot[i]; h.x = h_t[i]; h.y = h_li[i];
    }
    __syncwarp();
    if (lane == 0) {  // give the entries back, in order
      while (ld_volatile(&wsh->freed) != head) {}
      *reinterpret_cast<volatile uint32_t*>(&wsh->freed) = head + cnt;
    }
    // ---- shade
    bool cont = false, want_grad = false;
    uint32_t bad = 0, s = 0, k = 0;
    float4 n0, n1, n2;
    if (mine) {
      const float4* e = ring_entry(ws, slot);
      float4 Q0 = __ldcg(e);
      const float4 Q1 = __ldcg(e + cap), Q2 = __ldcg(e + 2 * cap);
      const uint32_t tag = __float_as_uint(Q0.w);
      s = tag & kStateMask;
      k = (tag >> kWaveKShift) + 1u;
      Q0.w = __uint_as_float(s);
      shade_vertex<GRAD>(sc, ws, io, k, Q0, Q1, Q2, h, s, cont, want_grad, bad, n0, n1, n2);
    }
    if (GRAD) {  // reverse-pass list: one atomic per warp
      const unsigned gm = __ballot_sync(kFull, want_grad);
      if (gm) {
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(&ws.ctl[kCtlGrad], (uint32_t)__popc(gm));
        base = __shfl_sync(kFull, base, 0);
        if (want_grad) ws.gradlist[base + __popc(gm & lt)] = s;
      }
    }
    // ---- the surviving paths' next rays -> global ring (reserve, write, publish in reservation order)
    const unsigned b = __ballot_sync(kFull, cont);
    const uint32_t nc = __popc(b);
    if (nc) {
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(&ws.ctl[kCtlWaveReserve], nc);
      base = __shfl_sync(kFull, base, 0);
      if (cont) {
        float4* e = ring_entry(ws, base + __popc(b & lt));
        n0.w = __uint_as_float(s | (k << kWaveKShift));   // segment k + 1, stored as k
        __stcg(e, n0); __stcg(e + cap, n1); __stcg(e + 2 * cap, n2);
        const uint32_t idx = base + __popc(b & lt);
        st_release(reinterpret_cast<uint32_t*>(ws.hits) + idx % (2u * ws.cap), idx / (2u * ws.cap) + 1u);
      }
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
template <bool GRAD>
__global__ void __launch_bounds__(kTraceBlock, 1) k_wave(DevScene sc, EvalWs ws, EvalIO io, uint32_t n) {
  static_assert(DR_SMEM_NODES == 0, "k_wave does not stage nodes in shared memory");
  extern __shared__ uint4 smem[];
  if (n == 0) return;
  // shared memory: one constant word | node stacks | triangle stacks | ring counters | ring
  SmemStack st{reinterpret_cast<uint2*>(smem + 1u) + threadIdx.x};
  SmemTriStack tst{st.base + (size_t)sc.stack_cap * kTraceBlock, nullptr};
  tst.base3 = reinterpret_cast<uint32_t*>(tst.base + (size_t)kTriStack * kTraceBlock - threadIdx.x) + threadIdx.x;
  uint32_t* tail = tst.base3 - threadIdx.x + (size_t)kTriStack * kTraceBlock;
  WaveShared* wsh = reinterpret_cast<WaveShared*>(tail);
  uint32_t* h_slot = tail + sizeof(WaveShared) / 4;
  uint32_t* h_t = h_slot + kHitCap;
  uint32_t* h_li = h_t + kHitCap;
  if (threadIdx.x == 0) {
    smem[0].x = 0x3F800000u;
    wsh->reserve = 0; wsh->pub = 0; wsh->head = 0; wsh->freed = 0;
  }
  __syncthreads();
  const uint32_t one = *(volatile uint32_t*)&smem[0].x;  // dr_traverse.cuh qmagic
  if (threadIdx.x >= (unsigned)kWaveTraceThreads) wave_shade_loop<GRAD>(sc, ws, io, n, wsh, h_slot, h_t, h_li);
  else wave_trace_loop(sc, ws, n, smem, st, tst, wsh, h_slot, h_t, h_li, one);
}

}  // namespace dr
