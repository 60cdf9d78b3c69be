// Host check of the scene builder and of the traversal building blocks (csrc/dr_bvh.cpp, csrc/dr_traverse.cuh),
// compiled and run by tests/test_bvh_host.py (no GPU).  It builds the BVH8 of a seeded mesh that mixes compact and
// long thin rotated triangles (what the reference pre-splitting of dr_bvh.cpp is for), then traces seeded rays through
// the host instantiation of the same node test / triangle test / work-mask state machine the kernel uses and compares
// every closest hit with a brute-force loop over all triangles (same triangle test, so t must agree bit for bit).
// Output: one line of key=value pairs.
#include <cstdio>
#include <cstdlib>
#include <random>
#include <set>
#include <vector>

#include "../paper_2605_08916_b200/csrc/dr_traverse.cuh"

using namespace dr;

struct HostMem {
  const BuiltBvh* b;
  void node(uint32_t i, uint4& w0, uint4& w1, uint4& w2, uint4& w3, uint4& w4) const {
    const uint4* p = reinterpret_cast<const uint4*>(&b->nodes[i]);
    w0 = p[0]; w1 = p[1]; w2 = p[2]; w3 = p[3]; w4 = p[4];
  }
  void tri(uint32_t li, float4& t0, float4& t1, float2& t2) const {
    const float4* p = reinterpret_cast<const float4*>(&b->tris[li]);
    t0 = p[0]; t1 = p[1]; t2 = make_float2(p[2].x, p[2].y);
  }
};
struct HostStack {
  uint2 e[64];
  void push(int sp, uint2 v) { e[sp] = v; }
  uint2 pop(int sp) const { return e[sp]; }
};

int main(int argc, char** argv) {
  const double budget = argc > 1 ? atof(argv[1]) : 1.0;
  const int n_tris = argc > 2 ? atoi(argv[2]) : 3000, n_rays = argc > 3 ? atoi(argv[3]) : 20000;
  std::mt19937 rng(7);
  std::uniform_real_distribution<float> U(0.f, 1.f);
  std::vector<float> v;
  std::vector<uint32_t> idx, mat;
  for (int t = 0; t < n_tris; ++t) {
    // every third triangle is a sliver: one long edge (up to 2), one short edge (down to 0.005), random orientation
    const bool sliver = t % 3 == 0;
    float c[3] = {4.f * U(rng), 4.f * U(rng), 4.f * U(rng)}, a[3], b[3];
    for (int k = 0; k < 3; ++k) { a[k] = U(rng) - 0.5f; b[k] = U(rng) - 0.5f; }
    const float la = sliver ? 2.0f : 0.3f, lb = sliver ? 0.005f + 0.02f * U(rng) : 0.3f;
    const uint32_t base = (uint32_t)(v.size() / 3);
    for (int k = 0; k < 3; ++k) v.push_back(c[k]);
    for (int k = 0; k < 3; ++k) v.push_back(c[k] + la * a[k]);
    for (int k = 0; k < 3; ++k) v.push_back(c[k] + lb * b[k]);
    idx.push_back(base); idx.push_back(base + 1); idx.push_back(base + 2);
    mat.push_back((uint32_t)(t % 5));
  }
  // two exact duplicates (tie rule: smaller original id) and one degenerate triangle (never hit)
  for (int k = 0; k < 3; ++k) idx.push_back(idx[k]);
  mat.push_back(1);
  idx.push_back(0); idx.push_back(0); idx.push_back(1);
  mat.push_back(2);
  const uint32_t nt = (uint32_t)(idx.size() / 3), nv = (uint32_t)(v.size() / 3);

  set_split_budget(budget);
  if (argc > 4) set_collapse(atoi(argv[4]) != 0, 1.0f, 0.4f);   // 1 = cost-optimal BVH2 -> BVH8 collapse (the default), 0 = greedy
  BuiltBvh b;
  build_bvh8(v.data(), nv, idx.data(), nt, mat.data(), b);

  // structure: every triangle referenced, ids / materials / edges stored as given, masks consistent
  std::set<uint32_t> seen;
  int bad_tri = 0;
  for (const TriPacked& tp : b.tris) {
    seen.insert(tp.id);
    if (tp.id >= nt || tp.mat != mat[tp.id]) { ++bad_tri; continue; }
    const float* a = &v[3 * idx[3 * tp.id]];
    const float* bb = &v[3 * idx[3 * tp.id + 1]];
    const float* c = &v[3 * idx[3 * tp.id + 2]];
    for (int k = 0; k < 3; ++k)
      if (tp.v0[k] != a[k] || tp.e1[k] != bb[k] - a[k] || tp.e2[k] != c[k] - a[k]) { ++bad_tri; break; }
  }
  int bad_node = 0;
  size_t tri_bits = 0, inner = 0;
  for (const NodeC& n : b.nodes) {
    if (n.imask32 != n.imask) ++bad_node;
    for (int s = 0; s < 8; ++s) {
      const uint32_t tb = (n.trimask >> (3 * s)) & 7u;
      if (tb != 0 && tb != 1 && tb != 3 && tb != 7) ++bad_node;     // unary count
      if (tb && ((n.imask >> s) & 1u)) ++bad_node;                    // a slot is a leaf or an internal child, not both
    }
    tri_bits += popc32(n.trimask);
    inner += popc32(n.imask);
  }
  if (tri_bits != b.tris.size() || inner + 1 != b.nodes.size()) ++bad_node;

  // closest hits: BVH8 traversal vs brute force
  HostMem mem{&b};
  int mismatch = 0, nhit = 0;
  unsigned long long nn = 0, ntt = 0;
  for (int i = 0; i < n_rays; ++i) {
    float o[3] = {-0.5f + 5.f * U(rng), -0.5f + 5.f * U(rng), -0.5f + 5.f * U(rng)}, d[3];
    float len = 0.f;
    do {
      len = 0.f;
      for (int k = 0; k < 3; ++k) { d[k] = 2.f * U(rng) - 1.f; len += d[k] * d[k]; }
    } while (len > 1.f || len < 1e-4f);
    for (int k = 0; k < 3; ++k) d[k] /= std::sqrt(len);
    if (i % 50 == 0) d[i % 3] = 0.f;  // axis-parallel components (the +-1e-20 nudge of trav_setup)
    TravRay ra, rb;
    trav_setup(ra, o[0], o[1], o[2], d[0], d[1], d[2]);
    rb = ra;
    HostStack st;
    uint32_t a_n = 0, a_t = 0;
    trav_closest_hit(mem, st, ra, &a_n, &a_t);
    nn += a_n; ntt += a_t;
    for (uint32_t li = 0; li < b.tris.size(); ++li) {
      float4 t0, t1; float2 t2;
      mem.tri(li, t0, t1, t2);
      tri_test(t0, t1, t2, li, rb);
    }
    if (ra.id != rb.id || f2u(ra.t) != f2u(rb.t)) ++mismatch;
    if (rb.id != 0xFFFFFFFFu) ++nhit;
  }
  std::printf("tris=%u refs=%zu referenced=%zu nodes=%zu depth=%u bad_tri=%d bad_node=%d rays=%d hits=%d mismatch=%d nodes_per_ray=%.2f tris_per_ray=%.2f\n",
              nt, b.tris.size(), seen.size(), b.nodes.size(), b.depth, bad_tri, bad_node, n_rays, nhit, mismatch,
              (double)nn / n_rays, (double)ntt / n_rays);
  return 0;
}
