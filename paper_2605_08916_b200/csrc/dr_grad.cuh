// Row a6 with next-event estimation: score g = grad p / (p + eps) of a listed state by a reverse sweep over its path.
// With emitter connections the contribution depends on the positions of the vertices, not only on directions (DESIGN.md
// Q21), so the sweep carries the adjoints of the ray that enters each vertex -- origin, direction and, for the MIS weight of
// an emitter found by the direction sample, the density of that direction.  The path is first replayed forwards from x and
// the recorded discrete decisions (triangle per segment, dielectric lobes, visibility bits: ws.rec), with vertex_fn<float>,
// the function the shading itself uses; then, last vertex first, the gradient of the scalar
//     Phi_k = sum_c lum_c T_k,c (C_k,c + W_k,c R_k+1,c) + o_bar . o_k+1 + d_bar . d_k+1 + pb_bar pb_k
// with respect to the vertex' ten inputs (o_k, d_k, u1, u2, v1, v2) is taken by three evaluations of vertex_fn<Du<4>>
// (T_k: throughput before the vertex, R_k+1: radiance per unit throughput from the later vertices, bars: adjoints of the
// next ray).  The u-part is the score of the vertex' coordinates, the (o, d)-part the adjoint handed to the vertex before.
// One thread = one listed state.  The oracle differentiates the same function with forward-mode dual numbers.
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

__device__ __forceinline__ void load_vertex(const DevScene& sc, uint32_t li, float3 d, VtxFrozen& f) {
  const float4 t0 = __ldg(&sc.tris[3 * li]), t1 = __ldg(&sc.tris[3 * li + 1]), t2 = __ldg(&sc.tris[3 * li + 2]);
  const float3 e1 = make_float3(t0.w, t1.x, t1.y), e2 = make_float3(t1.z, t1.w, t2.x);
  const uint32_t mi = __float_as_uint(t2.z);
  f.m0 = __ldg(&sc.mats[3 * mi]); f.m1 = __ldg(&sc.mats[3 * mi + 1]);
  f.kind = __float_as_uint(f.m0.x);
  f.v0 = xyz(t0);
  tri_frame(e1, e2, d, f.fr, f.dn);
}

// d Phi / d (four of the inputs).  mode 0: o.xyz, 1: d.xyz, 2: (u1, u2, v1, v2).  Also returns W and the visible C (values).
__device__ __noinline__ float4 vertex_phi_grad(const DevScene& sc, const VtxFrozen& f, float3 o, float3 d, float4 u, int mode, float3 lumT,
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
  vertex_fn<D>(sc, f.v0, f.fr, f.dn, f.m0, f.m1, f.kind, O, Dd, U1, U2, V1, V2, false, reflect, vo, hit, lj);
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

#ifndef DR_GRAD_MIN_BLOCKS
#define DR_GRAD_MIN_BLOCKS 6   // 80 registers: 1 / 3 / 4 / 6 blocks per SM: 6.12 / 5.90 / 5.64 / 5.32 ms per frame (configs[3] + NEE)
#endif
__global__ void __launch_bounds__(kGradBlock, DR_GRAD_MIN_BLOCKS) k_grad_nee(DevScene sc, EvalWs ws, EvalIO io) {
  const uint32_t idx = blockIdx.x * kGradBlock + threadIdx.x;
  if (idx == 0 && io.grad_ctr) atomicAdd(io.grad_ctr, (unsigned long long)ws.ctl[kCtlGrad]);
  if (idx >= ws.ctl[kCtlGrad]) return;
  const size_t cap = ws.cap;
  uint32_t rem = idx, bin = 15;   // the list is binned by the number of sampling vertices; longest paths first
  for (;; --bin) {
    const uint32_t c = ws.ctl[kCtlGradBin + bin];
    if (rem < c || bin == 0) break;
    rem -= c;
  }
  const uint32_t s = ws.gradlist[(size_t)bin * cap + rem];
  const float4 fp = io.f[s];
  const float inv_phat = 1.0f / (fp.w + kEps);
  const float4 hdr = ws.rec[s];
  const uint32_t info = __float_as_uint(hdr.x), term = __float_as_uint(hdr.z), nv = __float_as_uint(hdr.w);
  const float lum[3] = {0.2126f, 0.7152f, 0.0722f};
  // ---- forward replay: the ray entering every vertex, the throughput before it
  float3 O[kMaxPathLen + 1], Dv[kMaxPathLen + 1], Tk[kMaxPathLen + 1];
  float PB[kMaxPathLen + 1];
  uint32_t LI[kMaxPathLen + 1];
  const float4 x0 = io.x[s];
  {
    const V3<float> dc = camera_dir<float>(sc, x0.x, x0.y);
    O[1] = make_float3(sc.cam_pos[0], sc.cam_pos[1], sc.cam_pos[2]);
    Dv[1] = make_float3(dc.x, dc.y, dc.z);
    PB[1] = -1.f;
    Tk[1] = make_float3(1.f, 1.f, 1.f);
  }
  for (uint32_t k = 1; k <= nv; ++k) {
    LI[k] = __float_as_uint(ws.rec[(size_t)k * cap + s].w);
    VtxFrozen f;
    load_vertex(sc, LI[k], Dv[k], f);
    const float4 u = io.x[(size_t)k * io.stride + s];
    const V3<float> ov{O[k].x, O[k].y, O[k].z}, dv{Dv[k].x, Dv[k].y, Dv[k].z};
    VertexOut<float> vo;
    V3<float> hit;
    bool reflect = !((info >> k) & 1u);
    uint32_t lj = 0;
    vertex_fn<float>(sc, f.v0, f.fr, f.dn, f.m0, f.m1, f.kind, ov, dv, u.x, u.y, u.z, u.w, false, reflect, vo, hit, lj);
    O[k + 1] = make_float3(vo.o2.x, vo.o2.y, vo.o2.z);
    Dv[k + 1] = make_float3(vo.d2.x, vo.d2.y, vo.d2.z);
    PB[k + 1] = vo.pb_valid ? vo.pb : -1.f;
    Tk[k + 1] = make_float3(Tk[k].x * vo.W[0], Tk[k].y * vo.W[1], Tk[k].z * vo.W[2]);
  }
  // ---- what the path's last ray found
  float3 R = make_float3(0.f, 0.f, 0.f), ob = R, db = R;
  float pbb = 0.f;
  if (term == kMiss) {
    R = make_float3(sc.env[0], sc.env[1], sc.env[2]);
  } else if (term != kTermNone) {
    const float4 t0 = __ldg(&sc.tris[3 * term]), t1 = __ldg(&sc.tris[3 * term + 1]), t2 = __ldg(&sc.tris[3 * term + 2]);
    const float3 e1 = make_float3(t0.w, t1.x, t1.y), e2 = make_float3(t1.z, t1.w, t2.x);
    const uint32_t mi = __float_as_uint(t2.z);
    const float4 m1 = __ldg(&sc.mats[3 * mi + 1]), m2 = __ldg(&sc.mats[3 * mi + 2]);
    const float3 le = make_float3(m1.z, m1.w, m2.x);
    const float3 n = normalize3(cross3(e1, e2));
    const uint32_t K = nv + 1;
    if (dot3(Dv[K], n) < 0.f) {   // front face (the forward pass added T Le w_b)
      float wb = 1.f;
      if (PB[K] >= 0.f) {
        const float sL = lum[0] * Tk[K].x * le.x + lum[1] * Tk[K].y * le.y + lum[2] * Tk[K].z * le.z;
        const float4 go = emitter_weight_grad(sc, xyz(t0), n, O[K], Dv[K], PB[K], 0, &wb);
        const float4 gd = emitter_weight_grad(sc, xyz(t0), n, O[K], Dv[K], PB[K], 1, nullptr);
        ob = make_float3(sL * go.x, sL * go.y, sL * go.z);
        db = make_float3(sL * gd.x, sL * gd.y, sL * gd.z);
        pbb = sL * go.w;
      }
      R = make_float3(le.x * wb, le.y * wb, le.z * wb);
    }
  }
  // ---- reverse sweep
  bool bad = false;
  for (uint32_t k = nv; k >= 1; --k) {
    VtxFrozen f;
    load_vertex(sc, LI[k], Dv[k], f);
    f.reflect = !((info >> k) & 1u);
    f.vis = ((info >> (16u + k)) & 1u) != 0u;
    const float4 u = io.x[(size_t)k * io.stride + s];
    const float3 lumT = make_float3(lum[0] * Tk[k].x, lum[1] * Tk[k].y, lum[2] * Tk[k].z);
    float3 W, C;
    const float4 gu = vertex_phi_grad(sc, f, O[k], Dv[k], u, 2, lumT, R, ob, db, pbb, &W, &C);
    const float4 go = vertex_phi_grad(sc, f, O[k], Dv[k], u, 0, lumT, R, ob, db, pbb, nullptr, nullptr);
    const float4 gd = vertex_phi_grad(sc, f, O[k], Dv[k], u, 1, lumT, R, ob, db, pbb, nullptr, nullptr);
    const float4 g = make_float4(gu.x * inv_phat, gu.y * inv_phat, gu.z * inv_phat, gu.w * inv_phat);
    bad = bad || !(isfinite(g.x) && isfinite(g.y) && isfinite(g.z) && isfinite(g.w));
    io.g[(size_t)k * io.stride + s] = g;
    R = make_float3(C.x + W.x * R.x, C.y + W.y * R.y, C.z + W.z * R.z);
    ob = make_float3(go.x, go.y, go.z);
    db = make_float3(gd.x, gd.y, gd.z);
    pbb = 0.f;   // a vertex that samples does not use the density of the ray that reached it
  }
  {
    float ga = 0.f, gb = 0.f;
    if (db.x != 0.f || db.y != 0.f || db.z != 0.f) {   // the camera position is fixed: only the direction depends on the film point
      const V3<Du<2>> w = camera_dir<Du<2>>(sc, du_var<2>(x0.x, 0), du_var<2>(x0.y, 1));
      ga = (db.x * w.x.d[0] + db.y * w.y.d[0] + db.z * w.z.d[0]) * inv_phat;
      gb = (db.x * w.x.d[1] + db.y * w.y.d[1] + db.z * w.z.d[1]) * inv_phat;
    }
    bad = bad || !(isfinite(ga) && isfinite(gb));
    io.g[s] = make_float4(ga, gb, 0.f, 0.f);
  }
  if (bad) {  // Q18: a non-finite score makes the state a zero-contribution state
    io.f[s] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (uint32_t k = 0; k <= nv; ++k) io.g[(size_t)k * io.stride + s] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (io.nonfinite_ctr) atomicAdd(io.nonfinite_ctr, 1ull);
  }
}

}  // namespace dr
