// Host-side acceleration-structure build: binned-SAH BVH2, collapsed to a BVH8 and emitted breadth-first
// so that the top levels are contiguous (they are staged in shared memory by the traversal kernel).
// The paper uses a hardware ray-tracing pipeline; B200 has no RT cores, so the closest-hit
// query of row a4 runs in software over this structure.
#include <algorithm>
#include <cfloat>
#include <cmath>
#include <cstring>
#include <queue>

#include "dr_types.h"

namespace dr {
namespace {

struct Box {
  float lo[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, hi[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
  void grow(const float* p) { for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], p[a]); hi[a] = std::max(hi[a], p[a]); } }
  void grow(const Box& b) { for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], b.lo[a]); hi[a] = std::max(hi[a], b.hi[a]); } }
  float area() const {
    const float dx = hi[0] - lo[0], dy = hi[1] - lo[1], dz = hi[2] - lo[2];
    return dx < 0 ? 0.f : 2.f * (dx * dy + dy * dz + dz * dx);
  }
};

struct Node2 {
  Box box;
  uint32_t left = 0, right = 0;   // children (internal)
  uint32_t first = 0, count = 0;  // leaf range into `order`
};

// Empty child slots hold a far-away point box: the min/max slab test can never report a hit for it.
constexpr float kFar = 1e30f;
constexpr int kBins = 16;
constexpr uint32_t kLeafMax = 4;

struct Builder {
  const std::vector<Box>& tb;
  const std::vector<float>& cen;  // 3 per triangle
  std::vector<uint32_t> order;
  std::vector<Node2> nodes;

  Builder(const std::vector<Box>& b, const std::vector<float>& c) : tb(b), cen(c) {
    order.resize(b.size());
    for (uint32_t i = 0; i < order.size(); ++i) order[i] = i;
    nodes.reserve(2 * b.size());
  }

  uint32_t build(uint32_t first, uint32_t count) {
    const uint32_t me = (uint32_t)nodes.size();
    nodes.emplace_back();
    Box box, cb;
    for (uint32_t k = first; k < first + count; ++k) {
      box.grow(tb[order[k]]);
      cb.grow(&cen[3 * order[k]]);
    }
    nodes[me].box = box;
    nodes[me].first = first;
    nodes[me].count = count;
    if (count <= kLeafMax) return me;
    // binned SAH over the three axes
    float best_cost = FLT_MAX;
    int best_axis = -1, best_bin = -1;
    for (int a = 0; a < 3; ++a) {
      const float ext = cb.hi[a] - cb.lo[a];
      if (!(ext > 0.f)) continue;
      Box bb[kBins];
      uint32_t bc[kBins] = {0};
      const float scale = kBins / ext;
      for (uint32_t k = first; k < first + count; ++k) {
        int b = (int)((cen[3 * order[k] + a] - cb.lo[a]) * scale);
        b = std::min(std::max(b, 0), kBins - 1);
        bb[b].grow(tb[order[k]]);
        ++bc[b];
      }
      float la[kBins - 1], ra[kBins - 1];
      uint32_t lc[kBins - 1], rc[kBins - 1];
      Box acc; uint32_t n = 0;
      for (int b = 0; b < kBins - 1; ++b) { acc.grow(bb[b]); n += bc[b]; la[b] = acc.area(); lc[b] = n; }
      acc = Box(); n = 0;
      for (int b = kBins - 1; b > 0; --b) { acc.grow(bb[b]); n += bc[b]; ra[b - 1] = acc.area(); rc[b - 1] = n; }
      for (int b = 0; b < kBins - 1; ++b) {
        if (!lc[b] || !rc[b]) continue;
        const float cost = la[b] * lc[b] + ra[b] * rc[b];
        if (cost < best_cost) { best_cost = cost; best_axis = a; best_bin = b; }
      }
    }
    uint32_t mid;
    if (best_axis < 0) {  // all centroids coincide: split the range in half
      mid = first + count / 2;
    } else {
      const float ext = cb.hi[best_axis] - cb.lo[best_axis], scale = kBins / ext, lo = cb.lo[best_axis];
      auto it = std::partition(order.begin() + first, order.begin() + first + count, [&](uint32_t id) {
        int b = (int)((cen[3 * id + best_axis] - lo) * scale);
        b = std::min(std::max(b, 0), kBins - 1);
        return b <= best_bin;
      });
      mid = (uint32_t)(it - order.begin());
      if (mid == first || mid == first + count) mid = first + count / 2;
    }
    nodes[me].count = 0;
    const uint32_t l = build(first, mid - first);
    const uint32_t r = build(mid, first + count - mid);
    nodes[me].left = l;
    nodes[me].right = r;
    return me;
  }
};

}  // namespace

void build_bvh8(const float* verts, uint32_t nv, const uint32_t* idx, uint32_t nt, const uint32_t* tri_mat, BuiltBvh& out) {
  (void)nv;
  std::vector<Box> tb(nt);
  std::vector<float> cen(3 * (size_t)nt);
  Box scene;
  for (uint32_t t = 0; t < nt; ++t) {
    for (int k = 0; k < 3; ++k) tb[t].grow(&verts[3 * idx[3 * t + k]]);
    for (int a = 0; a < 3; ++a) cen[3 * t + a] = 0.5f * (tb[t].lo[a] + tb[t].hi[a]);
    scene.grow(tb[t]);
  }
  const float dx = scene.hi[0] - scene.lo[0], dy = scene.hi[1] - scene.lo[1], dz = scene.hi[2] - scene.lo[2];
  out.diag = nt ? std::sqrt(dx * dx + dy * dy + dz * dz) : 0.f;
  // Child boxes are inflated so that fp32 slab tests can never cull a triangle the exact test accepts:
  // slab rounding moves an entry/exit point by < 2e-7 * diag, the inflation is 20 times that.
  const float pad = 4e-6f * out.diag;
  out.nodes.clear();
  out.tris.clear();
  out.depth = 0;
  out.sah_cost = 0.f;
  if (!nt) {
    Node8 root;
    std::memset(&root, 0, sizeof(root));
    for (int i = 0; i < 8; ++i) {
      root.child[i] = kEmptyChild;
      for (int a = 0; a < 3; ++a) { root.lo[a][i] = kFar; root.hi[a][i] = kFar; }
    }
    out.nodes.push_back(root);
    return;
  }
  Builder b(tb, cen);
  b.build(0, nt);
  const std::vector<Node2>& n2 = b.nodes;

  // leaf-order triangle array
  out.tris.resize(nt);
  for (uint32_t k = 0; k < nt; ++k) {
    const uint32_t id = b.order[k];
    const float* a = &verts[3 * idx[3 * id]];
    const float* bb = &verts[3 * idx[3 * id + 1]];
    const float* c = &verts[3 * idx[3 * id + 2]];
    TriPacked& tp = out.tris[k];
    for (int x = 0; x < 3; ++x) { tp.v0[x] = a[x]; tp.e1[x] = bb[x] - a[x]; tp.e2[x] = c[x] - a[x]; }
    tp.id = id; tp.mat = tri_mat[id]; tp.pad = 0;
  }

  // collapse to BVH8, breadth-first
  struct Item { uint32_t n2; uint32_t depth; };
  std::queue<Item> q;
  q.push({0, 1});
  const float root_area = std::max(n2[0].box.area(), 1e-30f);
  double sah = 0.0;
  uint32_t next_index = 1;
  while (!q.empty()) {
    const Item it = q.front();
    q.pop();
    out.depth = std::max(out.depth, it.depth);
    uint32_t kids[8];
    int nk = 0;
    if (n2[it.n2].count) kids[nk++] = it.n2;  // root is itself a leaf
    else { kids[nk++] = n2[it.n2].left; kids[nk++] = n2[it.n2].right; }
    for (;;) {  // open the internal child with the largest area until 8 children
      if (nk == 8) break;
      int pick = -1;
      float pa = -1.f;
      for (int i = 0; i < nk; ++i)
        if (!n2[kids[i]].count && n2[kids[i]].box.area() > pa) { pa = n2[kids[i]].box.area(); pick = i; }
      if (pick < 0) break;
      const uint32_t p = kids[pick];
      kids[pick] = n2[p].left;
      kids[nk++] = n2[p].right;
    }
    Node8 node;
    std::memset(&node, 0, sizeof(node));
    for (int i = 0; i < 8; ++i) {
      if (i >= nk) {
        node.child[i] = kEmptyChild;
        for (int a = 0; a < 3; ++a) { node.lo[a][i] = kFar; node.hi[a][i] = kFar; }
        continue;
      }
      const Node2& c = n2[kids[i]];
      for (int a = 0; a < 3; ++a) { node.lo[a][i] = c.box.lo[a] - pad; node.hi[a][i] = c.box.hi[a] + pad; }
      if (c.count) {
        node.child[i] = kLeafBit | ((c.count - 1) << 27) | c.first;
        sah += (double)c.box.area() / root_area * c.count;
      } else {
        node.child[i] = next_index++;
        q.push({kids[i], it.depth + 1});
        sah += (double)c.box.area() / root_area;
      }
    }
    out.nodes.push_back(node);
  }
  out.sah_cost = (float)sah;
}

}  // namespace dr
