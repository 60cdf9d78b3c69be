// Row a6 with next-event estimation: score g = grad p / (p + eps) of every state with p > 0, by a reverse sweep over its path.
// With emitter connections the contribution depends on the positions of the vertices, not only on directions (DESIGN.md
// Q21), so the sweep carries the adjoints of the ray that enters each vertex -- origin, direction and, for the MIS weight of
// an emitter found by the direction sample, the density of that direction.  Last vertex first, the gradient of the scalar
//     Phi_k = sum_c lum_c T_k,c (C_k,c + W_k,c R_k+1,c) + o_bar . o_k+1 + d_bar . d_k+1 + pb_bar pb_k
// with respect to the vertex' ten inputs (o_k, d_k, u1, u2, v1, v2) is taken by evaluations of vertex_fn<Du<4>>, the function
// the shading itself uses with T = float (T_k: throughput before the vertex, R_k+1: radiance per unit throughput from the later
// vertices, bars: adjoints of the next ray).  The u-part is the score of the vertex' coordinates, the (o, d)-part the adjoint
// handed to the vertex before.  The oracle differentiates the same function with forward-mode dual numbers.
//
// Shape (profiles/r02g_grad_nee.md).  One thread per path ran with 12 of 32 lanes active (material kinds and connection
// outcomes differ from lane to lane) out of a 99 KB instruction footprint.  Now:
//   k_grad_nee_init           per state: what the path's last ray found (R and the adjoints of that ray) -> ws.adj; and the path's
//                             vertices go onto one list per (vertex index k, material kind of vertex k)
//   k_grad_nee_vertex<KIND>   k = L-1 .. 1, KIND = Lambert / dielectric / GGX: vertex k of every path that has one of that kind;
//                             every lane of a warp differentiates the same code, compiled for that kind alone
//   k_grad_nee_finish         Q18
// What the forward pass knew of the ray that reached a vertex (origin, direction, direction density, throughput) was recorded
// by the shading (record_vertex, dr_eval.cuh): there is no forward replay.  The adjoints wait in ws.adj between the launches.
#pragma once
#include "dr_eval.cuh"

namespace dr {

struct VtxFrozen {     // what the replay fixes for one vertex
  float3 v0;
  Frame fr;
  float dn;
  float4 m0, m1;
  uint32_t kind;
  bool reflect, vis;
};

// mi: the triangle's material index, known from the vertex record so that triangle and material arrive together
__device__ __forceinline__ void load_vertex(const DevScene& sc, uint32_t li, uint32_t mi, float3 d, VtxFrozen& f) {
  const float4 t0 = __ldg(&sc.tris[3 * li]), t1 = __ldg(&sc.tris[3 * li + 1]), t2 = __ldg(&sc.tris[3 * li + 2]);
  const float3 e1 = make_float3(t0.w, t1.x, t1.y), e2 = make_float3(t1.z, t1.w, t2.x);
  f.m0 = __ldg(&sc.mats[3 * mi]); f.m1 = __ldg(&sc.mats[3 * mi + 1]);
  f.kind = __float_as_uint(f.m0.x);
  f.v0 = xyz(t0);
  tri_frame(e1, e2, d, f.fr, f.dn);
}

// d Phi / d (four of the inputs) at a vertex of material KIND.  mode 0: o.xyz, 1: d.xyz, 2: (u1, u2, v1, v2).  Also returns W and
// the visible C (values).
template <int KIND>
__device__ __forceinline__ float4 vertex_phi_grad(const DevScene& sc, const VtxFrozen& f, float3 o, float3 d, float4 u, int mode, float3 lumT,
                                               float3 R, float3 ob, float3 db, float pbb, float3* W_out, float3* C_out) {
  typedef Du<4> D;
  V3<D> O{du_const<4>(o.x), du_const<4>(o.y), du_const<4>(o.z)}, Dd{du_const<4>(d.x), du_const<4>(d.y), du_const<4>(d.z)};
  D U1 = du_const<4>(u.x), U2 = du_const<4>(u.y), V1 = du_const<4>(u.z), V2 = du_const<4>(u.w);
  if (mode == 0) { O.x.d[0] = 1.f; O.y.d[1] = 1.f; O.z.d[2] = 1.f; }
  else if (mode == 1) { Dd.x.d[0] = 1.f; Dd.y.d[1] = 1.f; Dd.z.d[2] = 1.f; }
  else { U1.d[0] = 1.f; U2.d[1] = 1.f; V1.d[2] = 1.f; V2.d[3] = 1.f; }
  VertexOut<D> vo;
  V3<D> hit;
  bool reflect = f.reflect;
  uint32_t lj = 0;
  vertex_fn<D>(sc, f.v0, f.fr, f.dn, f.m0, f.m1, (uint32_t)KIND, O, Dd, U1, U2, V1, V2, false, reflect, vo, hit, lj);
  const bool conn = vo.nee_valid && f.vis;
  D phi = du_const<4>(0.f);
  const float lt[3] = {lumT.x, lumT.y, lumT.z}, Rr[3] = {R.x, R.y, R.z};
  float Wv[3], Cv[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    D term = vo.W[c] * Rr[c];
    Cv[c] = 0.f;
    if (conn) { const D cc = vo.fcos[c] * vo.lw[c]; term = term + cc; Cv[c] = cc.v; }
    phi = phi + term * lt[c];
    Wv[c] = vo.W[c].v;
  }
  if (vo.alive) {
    phi = phi + vo.o2.x * ob.x + vo.o2.y * ob.y + vo.o2.z * ob.z;
    phi = phi + vo.d2.x * db.x + vo.d2.y * db.y + vo.d2.z * db.z;
    if (vo.pb_valid) phi = phi + vo.pb * pbb;
  }
  if (W_out) *W_out = make_float3(Wv[0], Wv[1], Wv[2]);
  if (C_out) *C_out = make_float3(Cv[0], Cv[1], Cv[2]);
  return make_float4(phi.d[0], phi.d[1], phi.d[2], phi.d[3]);
}

// Emitter reached by the direction sample: w_b and its gradient with respect to (o.xyz, pb) [mode 0] or d.xyz [mode 1].
__device__ __noinline__ float4 emitter_weight_grad(const DevScene& sc, float3 v0, float3 n, float3 o, float3 d, float pb, int mode, float* w_out) {
  typedef Du<4> D;
  V3<D> O{du_const<4>(o.x), du_const<4>(o.y), du_const<4>(o.z)}, Dd{du_const<4>(d.x), du_const<4>(d.y), du_const<4>(d.z)};
  D PB = du_const<4>(pb);
  if (mode == 0) { O.x.d[0] = 1.f; O.y.d[1] = 1.f; O.z.d[2] = 1.f; PB.d[3] = 1.f; }
  else { Dd.x.d[0] = 1.f; Dd.y.d[1] = 1.f; Dd.z.d[2] = 1.f; }
  const D w = emitter_weight<D>(sc, v0, n, O, Dd, PB, true);
  if (w_out) *w_out = w.v;
  return make_float4(w.d[0], w.d[1], w.d[2], w.d[3]);
}

constexpr int kGradVertexBlock = 128;
constexpr uint32_t kRecLiMask = 0x3FFFFFFFu;   // ws.rec[k].w = triangle (leaf order) | material kind << 30
// list of the paths whose vertex k has material `kind`: entries ws.gradlist[(3 k + kind) * cap ...], count ws.ctl[kCtlGradKind + 3 k + kind]
__device__ __forceinline__ uint32_t grad_list(uint32_t k, uint32_t kind) { return 3u * k + kind; }

// Per state, in index order (the shading wrote f, the header ws.rec[s], the vertex records and the vertex kinds ws.pinfo[s] of
// every finished path): the path's vertices go onto the (k, kind) lists -- counted per block in shared memory, one atomic per
// block and list -- and what the path's last ray found, R (radiance per unit throughput) and the adjoints of that ray, goes
// into ws.adj.
constexpr int kGradInitBlock = 256;
constexpr int kGradLists = 3 * kMaxPathLen;
__global__ void __launch_bounds__(kGradInitBlock) k_grad_nee_init(DevScene sc, EvalWs ws, EvalIO io, uint32_t n) {
  __shared__ uint32_t s_cnt[kGradInitBlock / 32][kGradLists];   // entries of warp w for list j; then their offset in the list
  const uint32_t s = blockIdx.x * kGradInitBlock + threadIdx.x;
  const size_t cap = ws.cap;
  const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5, lt = (1u << lane) - 1u;
  const bool listed = s < n && io.f[s].w > 0.f;   // finish_path: p > 0
  uint32_t nv = 0, term = kTermNone, kinds = 0;
  if (listed) {
    const float4 hdr = ws.rec[s];
    term = __float_as_uint(hdr.z); nv = __float_as_uint(hdr.w);
    kinds = ws.pinfo[s];
  }
  {
    const unsigned lm = __ballot_sync(0xFFFFFFFFu, listed);
    if (lane == 0 && lm && io.grad_ctr) atomicAdd(io.grad_ctr, (unsigned long long)__popc(lm));
  }
  for (uint32_t j = lane; j < (uint32_t)kGradLists; j += 32) s_cnt[wid][j] = 0;
  __syncwarp();
  const uint32_t kmax = __reduce_max_sync(0xFFFFFFFFu, nv);
  for (uint32_t k = 1; k <= kmax; ++k) {
    const uint32_t kind = k <= nv ? ((kinds >> (2u * (k - 1u))) & 3u) : 3u;
#pragma unroll
    for (uint32_t q = 0; q < 3; ++q) {
      const unsigned m = __ballot_sync(0xFFFFFFFFu, kind == q);
      if (lane == 0) s_cnt[wid][grad_list(k, q)] = __popc(m);
    }
  }
  __syncthreads();
  if (threadIdx.x < kGradLists) {   // one thread per list: the block's entries, one atomic, the warps' offsets
    uint32_t tot = 0;
    for (int w = 0; w < kGradInitBlock / 32; ++w) tot += s_cnt[w][threadIdx.x];
    uint32_t base = tot ? atomicAdd(&ws.ctl[kCtlGradKind + threadIdx.x], tot) : 0u;
    for (int w = 0; w < kGradInitBlock / 32; ++w) { const uint32_t c = s_cnt[w][threadIdx.x]; s_cnt[w][threadIdx.x] = base; base += c; }
  }
  __syncthreads();
  for (uint32_t k = 1; k <= kmax; ++k) {
    const uint32_t kind = k <= nv ? ((kinds >> (2u * (k - 1u))) & 3u) : 3u;
    const unsigned m = __ballot_sync(0xFFFFFFFFu, kind < 3u) & __match_any_sync(0xFFFFFFFFu, kind);   // the lanes of my kind
    if (kind < 3u) ws.gradlist[(size_t)grad_list(k, kind) * cap + s_cnt[wid][grad_list(k, kind)] + __popc(m & lt)] = s;
  }
  if (!listed) return;
  float3 R = make_float3(0.f, 0.f, 0.f), ob = R, db = R;
  float pbb = 0.f;
  if (term == kMiss) {
    R = make_float3(sc.env[0], sc.env[1], sc.env[2]);
  } else if (term != kTermNone) {
    const float4* vr = ws.vrec + vrec_at(ws, nv + 1, s);   // the emitter hit was recorded as vertex nv + 1
    const float4 rD = vr[0], rO = vr[1], rT = vr[2];
    const float4 t0 = __ldg(&sc.tris[3 * term]), t1 = __ldg(&sc.tris[3 * term + 1]), t2 = __ldg(&sc.tris[3 * term + 2]);
    const float3 e1 = make_float3(t0.w, t1.x, t1.y), e2 = make_float3(t1.z, t1.w, t2.x);
    const uint32_t mi = __float_as_uint(t2.z);
    const float4 m1 = __ldg(&sc.mats[3 * mi + 1]), m2 = __ldg(&sc.mats[3 * mi + 2]);
    const float3 le = make_float3(m1.z, m1.w, m2.x);
    const float3 nrm = normalize3(cross3(e1, e2));
    const float3 o = xyz(rO), d = xyz(rD);
    const float pb = rO.w;
    if (dot3(d, nrm) < 0.f) {   // front face (the forward pass added T Le w_b)
      float wb = 1.f;
      if (pb >= 0.f) {
        const float sL = 0.2126f * rT.x * le.x + 0.7152f * rT.y * le.y + 0.0722f * rT.z * le.z;
        const float4 go = emitter_weight_grad(sc, xyz(t0), nrm, o, d, pb, 0, &wb);
        const float4 gd = emitter_weight_grad(sc, xyz(t0), nrm, o, d, pb, 1, nullptr);
        ob = make_float3(sL * go.x, sL * go.y, sL * go.z);
        db = make_float3(sL * gd.x, sL * gd.y, sL * gd.z);
        pbb = sL * go.w;
      }
      R = make_float3(le.x * wb, le.y * wb, le.z * wb);
    }
  }
  float4* aj = ws.adj + 3 * (size_t)s;
  aj[0] = make_float4(R.x, R.y, R.z, ob.x);
  aj[1] = make_float4(ob.y, ob.z, db.x, db.y);
  aj[2] = make_float4(db.z, pbb, 0.f, 0.f);   // .w: "score not finite" flag of the sweep
}

#ifndef DR_GRAD_MIN_BLOCKS
#define DR_GRAD_MIN_BLOCKS 4
#endif
#ifndef DR_GRAD_LAMBERT_SPLIT
#define DR_GRAD_LAMBERT_SPLIT 1
#endif
#ifndef DR_GRAD_GGX_SPLIT
#define DR_GRAD_GGX_SPLIT 1
#endif
// Vertex k of every path whose vertex k has material KIND (0 Lambert, 1 dielectric, 2 GGX).
// Phi depends on the ray (o, d) through the hit point h = o + t d on the frozen plane, t = ((v0 - o).n) / (d.n), and -- for a
// dielectric or GGX vertex only -- on d itself.  With P = I - d n^T / (d.n):  dPhi/do = P^T dPhi/dh,  dPhi/dd = t P^T dPhi/dh
// + (dPhi/dd at fixed h).  So a Lambert vertex needs no pass over d (dPhi/dd = t dPhi/do), and a dielectric vertex, which makes
// no connection and has weight one, needs only the Jacobian of its outgoing direction.
template <int KIND>
__device__ __forceinline__ void grad_vertex(const DevScene& sc, const EvalWs& ws, const EvalIO& io, uint32_t k, uint32_t idx) {
  const size_t cap = ws.cap;
  const uint32_t s = ws.gradlist[(size_t)grad_list(k, KIND) * cap + idx];
  const float4* vr = ws.vrec + vrec_at(ws, k, s);
  float4* aj = ws.adj + 3 * (size_t)s;
  const float4 rD = vr[0], rO = vr[1], rT = vr[2];
  const uint32_t info = __float_as_uint(ws.rec[s].x);
  const float4 a0 = aj[0], a1 = aj[1], a2 = aj[2];
  float3 R = make_float3(a0.x, a0.y, a0.z), ob = make_float3(a0.w, a1.x, a1.y), db = make_float3(a1.z, a1.w, a2.x);
  const float pbb = a2.y;
  const float3 o = xyz(rO), d = xyz(rD);
  VtxFrozen f;
  load_vertex(sc, __float_as_uint(rD.w) & kRecLiMask, __float_as_uint(rT.w), d, f);
  f.reflect = !((info >> k) & 1u);
  f.vis = ((info >> (16u + k)) & 1u) != 0u;
  const float inv_phat = 1.0f / (io.f[s].w + kEps);
  const float side = f.dn < 0.f ? 1.f : -1.f;
  const float3 n = f.fr.nf * side;
  const float dnn = dot3(d, n);
  const float tp = dot3(f.v0 - o, n) / dnn;
  float3 W = make_float3(1.f, 1.f, 1.f), C = make_float3(0.f, 0.f, 0.f);
  float4 gu = make_float4(0.f, 0.f, 0.f, 0.f), go, gd;
  if (KIND == 1) {
    const float c = dot3(d, ob) / dnn;
    go = make_float4(ob.x - n.x * c, ob.y - n.y * c, ob.z - n.z * c, 0.f);   // P^T o_bar  (o2 = h + const)
    const float eta = f.dn < 0.f ? f.m1.x : 1.0f / f.m1.x;
    const V3<Du<3>> di{du_var<3>(d.x, 0), du_var<3>(d.y, 1), du_var<3>(d.z, 2)};
    const V3<Du<3>> w = dielectric_dir<Du<3>>(f.fr, eta, f.reflect, di);
    gd = make_float4(tp * go.x + (db.x * w.x.d[0] + db.y * w.y.d[0] + db.z * w.z.d[0]),
                     tp * go.y + (db.x * w.x.d[1] + db.y * w.y.d[1] + db.z * w.z.d[1]),
                     tp * go.z + (db.x * w.x.d[2] + db.y * w.y.d[2] + db.z * w.z.d[2]), 0.f);
  } else if (KIND == 0 && DR_GRAD_LAMBERT_SPLIT) {
    // Lambert: the direction sample depends on (u1, u2) alone (two tangents), the connection on (h, v1, v2) alone (five): each
    // part is differentiated once with just its own tangents, instead of the whole vertex twice with four
    const float4 u = io.x[(size_t)k * io.stride + s];
    const float3 lumT = make_float3(0.2126f * rT.x, 0.7152f * rT.y, 0.0722f * rT.z);
    W = make_float3(f.m0.y, f.m0.z, f.m0.w);
    float3 gh = ob;                                             // o2 = h + const
    {
      typedef Du<5> D;
      V3<D> H;                                                  // h = o + t d, as the shading computes it
      H.x = du_var<5>(o.x + d.x * tp, 0); H.y = du_var<5>(o.y + d.y * tp, 1); H.z = du_var<5>(o.z + d.z * tp, 2);
      const V3<D> Dc{du_const<5>(d.x), du_const<5>(d.y), du_const<5>(d.z)};
      VertexOut<D> vo;
      uint32_t lj = 0;
      nee_connect<D>(sc, f.fr, f.m0, f.m1, 0u, Dc, H, du_var<5>(u.z, 3), du_var<5>(u.w, 4), vo, lj);
      if (vo.nee_valid && f.vis) {
        const D c0 = vo.fcos[0] * vo.lw[0], c1 = vo.fcos[1] * vo.lw[1], c2 = vo.fcos[2] * vo.lw[2];
        C = make_float3(c0.v, c1.v, c2.v);
        const D phi = c0 * lumT.x + c1 * lumT.y + c2 * lumT.z;
        gh = make_float3(gh.x + phi.d[0], gh.y + phi.d[1], gh.z + phi.d[2]);
        gu.z = phi.d[3]; gu.w = phi.d[4];
      }
    }
    {
      const V3<Du<2>> w = lambert_dir<Du<2>>(f.fr, du_var<2>(u.x, 0), du_var<2>(u.y, 1));
      const Du<2> pb = sqrt_t(1.0f - du_var<2>(u.x, 0)) * kInvPi;
      gu.x = (db.x * w.x.d[0] + db.y * w.y.d[0] + db.z * w.z.d[0]) + pb.d[0] * pbb;
      gu.y = (db.x * w.x.d[1] + db.y * w.y.d[1] + db.z * w.z.d[1]) + pb.d[1] * pbb;
    }
    const float c = dot3(d, gh) / dnn;
    go = make_float4(gh.x - n.x * c, gh.y - n.y * c, gh.z - n.z * c, 0.f);   // P^T dPhi/dh
    gd = make_float4(tp * go.x, tp * go.y, tp * go.z, 0.f);
  } else if (KIND == 2 && DR_GRAD_GGX_SPLIT) {
    // GGX: Phi = Phi_conn(h, d, v1, v2) + Phi_dir(d, u1, u2) + o2 . o_bar.  The connection is differentiated in two passes of four
    // tangents, (h, v1) and (d, v2), the direction sample once over (d, u1, u2): three passes of the whole vertex before
    const float4 u = io.x[(size_t)k * io.stride + s];
    const float3 lumT = make_float3(0.2126f * rT.x, 0.7152f * rT.y, 0.0722f * rT.z);
    const float3 h = make_float3(o.x + d.x * tp, o.y + d.y * tp, o.z + d.z * tp);   // as the shading computes it
    float3 gh = make_float3(0.f, 0.f, 0.f), gdd = gh;      // dPhi/dh, dPhi/dd at fixed h
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
      typedef Du<4> D;
      V3<D> H{du_const<4>(h.x), du_const<4>(h.y), du_const<4>(h.z)}, Dd{du_const<4>(d.x), du_const<4>(d.y), du_const<4>(d.z)};
      D V1 = du_const<4>(u.z), V2 = du_const<4>(u.w);
      if (pass == 0) { H.x.d[0] = 1.f; H.y.d[1] = 1.f; H.z.d[2] = 1.f; V1.d[3] = 1.f; }
      else { Dd.x.d[0] = 1.f; Dd.y.d[1] = 1.f; Dd.z.d[2] = 1.f; V2.d[3] = 1.f; }
      VertexOut<D> vo;
      uint32_t lj = 0;
      nee_connect<D>(sc, f.fr, f.m0, f.m1, 2u, Dd, H, V1, V2, vo, lj);
      if (vo.nee_valid && f.vis) {
        const D c0 = vo.fcos[0] * vo.lw[0], c1 = vo.fcos[1] * vo.lw[1], c2 = vo.fcos[2] * vo.lw[2];
        const D phi = c0 * lumT.x + c1 * lumT.y + c2 * lumT.z;
        if (pass == 0) { C = make_float3(c0.v, c1.v, c2.v); gh = make_float3(phi.d[0], phi.d[1], phi.d[2]); gu.z = phi.d[3]; }
        else { gdd = make_float3(phi.d[0], phi.d[1], phi.d[2]); gu.w = phi.d[3]; }
      }
    }
    {
      typedef Du<5> D;
      const V3<D> Dd{du_var<5>(d.x, 0), du_var<5>(d.y, 1), du_var<5>(d.z, 2)};
      VertexOut<D> vo;
      vo.alive = true; vo.pb_valid = false; vo.pb = du_const<5>(0.f);
      ggx_sample<D>(sc, f.fr, f.m0, f.m1, Dd, du_var<5>(u.x, 3), du_var<5>(u.y, 4), vo);
      W = make_float3(vo.W[0].v, vo.W[1].v, vo.W[2].v);
      if (vo.alive) {
        D phi = vo.W[0] * (lumT.x * R.x) + vo.W[1] * (lumT.y * R.y) + vo.W[2] * (lumT.z * R.z);
        phi = phi + vo.d2.x * db.x + vo.d2.y * db.y + vo.d2.z * db.z;
        if (vo.pb_valid) phi = phi + vo.pb * pbb;
        gdd = make_float3(gdd.x + phi.d[0], gdd.y + phi.d[1], gdd.z + phi.d[2]);
        gu.x = phi.d[3]; gu.y = phi.d[4];
        gh = gh + ob;                                        // o2 = h + const
      }
    }
    const float c = dot3(d, gh) / dnn;
    go = make_float4(gh.x - n.x * c, gh.y - n.y * c, gh.z - n.z * c, 0.f);   // P^T dPhi/dh
    gd = make_float4(tp * go.x + gdd.x, tp * go.y + gdd.y, tp * go.z + gdd.z, 0.f);
  } else {
    const float4 u = io.x[(size_t)k * io.stride + s];
    const float3 lumT = make_float3(0.2126f * rT.x, 0.7152f * rT.y, 0.0722f * rT.z);
    // one copy of the differentiated vertex in the code, run two (Lambert) or three times: everything stays in registers
#pragma unroll 1
    for (int pass = 0; pass < (KIND == 0 ? 2 : 3); ++pass) {
      float3 Wp, Cp;
      const float4 r = vertex_phi_grad<KIND>(sc, f, o, d, u, pass == 0 ? 2 : pass - 1, lumT, R, ob, db, pbb, &Wp, &Cp);
      if (pass == 0) { gu = r; W = Wp; C = Cp; }
      else if (pass == 1) go = r;
      else gd = r;
    }
    if (KIND == 0) gd = make_float4(tp * go.x, tp * go.y, tp * go.z, 0.f);
  }
  const float4 g = make_float4(gu.x * inv_phat, gu.y * inv_phat, gu.z * inv_phat, gu.w * inv_phat);
  bool bad = !(isfinite(g.x) && isfinite(g.y) && isfinite(g.z) && isfinite(g.w));
  io.g[(size_t)k * io.stride + s] = g;
  R = make_float3(C.x + W.x * R.x, C.y + W.y * R.y, C.z + W.z * R.z);
  ob = make_float3(go.x, go.y, go.z);
  db = make_float3(gd.x, gd.y, gd.z);
  if (k > 1u) {   // a vertex that samples does not use the density of the ray that reached it: pb_bar = 0
    aj[0] = make_float4(R.x, R.y, R.z, ob.x);
    aj[1] = make_float4(ob.y, ob.z, db.x, db.y);
    aj[2] = make_float4(db.z, 0.f, 0.f, (bad || a2.w != 0.f) ? 1.f : 0.f);
  } else {        // the camera: its position is fixed, only the direction depends on the film point
    float ga = 0.f, gb = 0.f;
    if (db.x != 0.f || db.y != 0.f || db.z != 0.f) {
      const float4 x0 = io.x[s];
      const V3<Du<2>> w = camera_dir<Du<2>>(sc, du_var<2>(x0.x, 0), du_var<2>(x0.y, 1));
      ga = (db.x * w.x.d[0] + db.y * w.y.d[0] + db.z * w.z.d[0]) * inv_phat;
      gb = (db.x * w.x.d[1] + db.y * w.y.d[1] + db.z * w.z.d[1]) * inv_phat;
    }
    bad = bad || !(isfinite(ga) && isfinite(gb));
    io.g[s] = make_float4(ga, gb, 0.f, 0.f);
    if (bad || a2.w != 0.f) aj[2] = make_float4(0.f, 0.f, 0.f, 1.f);
  }
}

// One launch per vertex index: the blocks are dealt to the three lists of that index in turn (list lengths are known on the
// device only: the grid covers the worst case and the blocks past the end leave at once).
__global__ void __launch_bounds__(kGradVertexBlock, DR_GRAD_MIN_BLOCKS) k_grad_nee_vertex(DevScene sc, EvalWs ws, EvalIO io, uint32_t k) {
  const uint32_t c0 = ws.ctl[kCtlGradKind + grad_list(k, 0)], c1 = ws.ctl[kCtlGradKind + grad_list(k, 1)], c2 = ws.ctl[kCtlGradKind + grad_list(k, 2)];
  const uint32_t nb0 = (c0 + kGradVertexBlock - 1) / kGradVertexBlock, nb2 = (c2 + kGradVertexBlock - 1) / kGradVertexBlock;
  uint32_t b = blockIdx.x;
  // GGX first (the longest blocks), then Lambert, then dielectric
  if (b < nb2) { const uint32_t idx = b * kGradVertexBlock + threadIdx.x; if (idx < c2) grad_vertex<2>(sc, ws, io, k, idx); return; }
  b -= nb2;
  if (b < nb0) { const uint32_t idx = b * kGradVertexBlock + threadIdx.x; if (idx < c0) grad_vertex<0>(sc, ws, io, k, idx); return; }
  b -= nb0;
  const uint32_t idx = b * kGradVertexBlock + threadIdx.x;
  if (idx < c1) grad_vertex<1>(sc, ws, io, k, idx);
}

// Q18: a non-finite score makes the state a zero-contribution state
__global__ void __launch_bounds__(kGradBlock) k_grad_nee_finish(DevScene sc, EvalWs ws, EvalIO io, uint32_t n) {
  const uint32_t s = blockIdx.x * kGradBlock + threadIdx.x;
  if (s >= n || !(io.f[s].w > 0.f) || ws.adj[3 * (size_t)s + 2].w == 0.f) return;
  const uint32_t nv = __float_as_uint(ws.rec[s].w);
  io.f[s] = make_float4(0.f, 0.f, 0.f, 0.f);
  for (uint32_t k = 0; k <= nv; ++k) io.g[(size_t)k * io.stride + s] = make_float4(0.f, 0.f, 0.f, 0.f);
  if (io.nonfinite_ctr) atomicAdd(io.nonfinite_ctr, 1ull);
}

}  // namespace dr
